// mm_api.cu -- host side of the C-ABI in include/mm.h: argument checks, workspace carving and
// kernel launches.  No arithmetic of the method runs here; there is no CPU fallback.
#include "../../include/mm.h"
#include "mm_kernels.cuh"
#include "mm_tm14.cuh"
#include "mm_batch5.cuh"

#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

using namespace mm;

namespace {

constexpr int kNT5 = 128;               // 5-moment cells per block
constexpr int kRateNT = 256;

// The 14-moment step kernel (mm_tm14.cuh) runs one block of Mom<ZS>::NW warps per SM; a warp is one
// work item (strip x row chunk).
constexpr size_t kSmemGen = Mom<false>::smem_bytes, kSmemZS = Mom<true>::smem_bytes;
constexpr int kWarpsGen = Mom<false>::NW, kWarpsZS = Mom<true>::NW;
static_assert(kSmemGen <= 227 * 1024 && kSmemZS <= 227 * 1024, "strip buffers exceed the shared memory of an SM");

thread_local char g_cuda_msg[256] = "";

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Layout {
    int nm, pitch, rows;
    size_t plane, state_bytes, off_ctrl, off_bc, off_tab, off_hist, off_u0, off_u1, off_w0, off_w1, total;
};

bool make_layout(const mm_grid* g, Layout* L)
{
    if (!g) return false;
    if (g->system != MM_SYS5_1D && g->system != MM_SYS14_2D) return false;
    if (g->nx < 1 || g->ny < 1 || !(g->x1 > g->x0)) return false;
    if (g->system == MM_SYS5_1D && g->ny != 1) return false;
    if (g->system == MM_SYS14_2D && !(g->y1 > g->y0)) return false;
    L->nm = g->system;
    L->pitch = (int)align_up((size_t)g->nx + 4, 16);
    L->rows = g->ny + 4;
    L->plane = (size_t)L->pitch * L->rows;
    L->state_bytes = align_up(L->plane * L->nm * sizeof(double), 256);
    L->off_ctrl = 0;
    L->off_bc = align_up(sizeof(Ctrl), 256);
    L->off_tab = L->off_bc + align_up(sizeof(BcTable), 256);
    L->off_hist = L->off_tab + align_up(AbTable::kDoubles * sizeof(double), 256);
    L->off_u0 = L->off_hist + align_up((size_t)kDtHistory * sizeof(double), 256);
    L->off_u1 = L->off_u0 + L->state_bytes;
    // the 14-moment system keeps the primitives W(U) of both copies beside them (mm_tm14.cuh)
    L->off_w0 = L->off_u1 + L->state_bytes;
    L->off_w1 = L->off_w0 + (L->nm == 14 ? L->state_bytes : 0);
    L->total = L->off_w1 + (L->nm == 14 ? L->state_bytes : 0);
    return true;
}

// Strips are kSW cells wide; rows are cut into nchunks chunks so that the nstrips * nchunks items (one
// per warp) fill whole waves of the `slots` resident warps.  A chunk of n rows costs n + ~0.8 row
// passes (one extra y-interface row and four extra row conversions).
void choose_decomposition(int nx, int ny, int slots, int* nstrips, int* nchunks)
{
    const int ns = (nx + kSW - 1) / kSW;
    double best = 1e300;
    int bestc = 1;
    for (int c = 1; c <= ny; ++c) {
        const int rows = (ny + c - 1) / c;
        const long long waves = ((long long)ns * c + slots - 1) / slots;
        const double cost = (double)waves * (rows + 0.8);
        if (cost < best * (1.0 - 1e-9)) { best = cost; bestc = c; }
    }
    *nstrips = ns; *nchunks = bestc;
}

}  // namespace

struct mm_solver {
    mm_grid grid;
    Layout L;
    Params p;
    cudaStream_t stream;
    char* ws;
    Ctrl* ctrl;
    BcTable* bc;
    double* U[2];
    double* W[2];       // 14-moment: primitives of U[0], U[1] (nullptr for the 5-moment system)
    int cur;            // buffer holding the current state
    int slot;           // accumulator slot holding the current state's CFL reduction
    int has_state;
    long long hist_first;   // dt history is valid for steps >= hist_first (mm_set_clock moves it)
    long long launches;
    int nstrips, nchunks[2];   // 14-moment work decomposition (mm_tm14.cuh): [general, z-symmetric]
    int time_scheme;        // MM_TIME_EULER | MM_TIME_MIDPOINT
    int zsym;               // state and boundary data have no z-odd moment: fast path applies
    int allow_fast;         // mm_set_fast_path
    int sms;
    bool profiling;
    std::vector<cudaEvent_t> ev;   // start/stop pairs around the step kernel while profiling
};

namespace {

int cuda_fail(cudaError_t e, const char* what)
{
    snprintf(g_cuda_msg, sizeof g_cuda_msg, "CUDA error in %s: %s", what, cudaGetErrorString(e));
    return MM_ECUDA;
}
#define MM_CUDA(call)                                                        \
    do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)
#define MM_LAUNCHED(s, what)                                                 \
    do { (s)->launches++; cudaError_t e_ = cudaGetLastError();               \
         if (e_ != cudaSuccess) return cuda_fail(e_, what); } while (0)

template <int NM>
int launch_ghost(mm_solver* s, const StepCtl& sc, int finalize)
{
    const int n = 4 * s->p.ny + (NM == 5 ? 0 : 4 * s->p.nx);
    const int nt = 128, nb = (n + nt - 1) / nt;
    k_ghost<NM><<<nb, nt, 0, s->stream>>>(s->p, NM == 14 ? s->W[s->cur] : s->U[s->cur], s->bc, s->ctrl, s->slot, sc,
                                          finalize, (double*)(s->ws + s->L.off_hist), NM == 14);
    MM_LAUNCHED(s, "k_ghost");
    return MM_OK;
}

// one pass of the fused step kernel: U[out] = B - dt_scale dt div F(U[in]) + source
int launch_pass(mm_solver* s, int in, int out, const double* base, double dt_scale, int do_rate)
{
    if (s->L.nm == 5) {
        const int nb = (s->p.nx + kNT5 - 1) / kNT5;
        k_step5<kNT5><<<nb, kNT5, 0, s->stream>>>(s->p, s->U[in], s->U[out], s->ctrl, s->slot ^ 1, base, dt_scale, do_rate);
        MM_LAUNCHED(s, "k_step5");
    } else {
        const int fast = s->zsym && s->allow_fast;
        const int items = s->nstrips * s->nchunks[fast];
        const bool ext = base != nullptr || dt_scale != 1.0 || !do_rate || s->p.source_scheme != 0;
#define MM_LAUNCH_TM(ZSV, EXTV)                                                                      \
    k_step14_tm<ZSV, EXTV><<<(items + Mom<ZSV>::NW - 1) / Mom<ZSV>::NW, 32 * Mom<ZSV>::NW,             \
                             Mom<ZSV>::smem_bytes, s->stream>>>(                                       \
        s->p, s->W[in], s->U[in], s->W[out], s->U[out], s->ctrl, s->slot ^ 1, s->nstrips, s->nchunks[fast], base, dt_scale, do_rate)
        if (fast) { if (ext) MM_LAUNCH_TM(true, true); else MM_LAUNCH_TM(true, false); }
        else { if (ext) MM_LAUNCH_TM(false, true); else MM_LAUNCH_TM(false, false); }
#undef MM_LAUNCH_TM
        MM_LAUNCHED(s, "k_step14_tm");
    }
    return MM_OK;
}

template <int NM>
int launch_step_nm(mm_solver* s, const StepCtl& sc, cudaEvent_t e0, cudaEvent_t e1)
{
    int rc;
    if ((rc = launch_ghost<NM>(s, sc, 1))) return rc;            // ghosts of U^n, dt from its CFL rate
    if (e0) MM_CUDA(cudaEventRecord(e0, s->stream));
    const int a = s->cur, b = s->cur ^ 1;
    if (s->time_scheme == MM_TIME_MIDPOINT) {
        // U' = U^n + dt/2 L(U^n) -> b;  ghosts of U';  U^{n+1} = U^n + dt L(U') -> a, in place
        if ((rc = launch_pass(s, a, b, nullptr, 0.5, 0))) return rc;
        s->cur = b;
        StepCtl none = {0, 0.0, -1.0};
        rc = launch_ghost<NM>(s, none, 0);
        s->cur = a;
        if (rc) return rc;
        if ((rc = launch_pass(s, b, a, s->U[a], 1.0, 1))) return rc;
    } else {
        if ((rc = launch_pass(s, a, b, nullptr, 1.0, 1))) return rc;
        s->cur = b;
    }
    if (e1) MM_CUDA(cudaEventRecord(e1, s->stream));
    s->slot ^= 1;
    return MM_OK;
}

int launch_step(mm_solver* s, const StepCtl& sc)
{
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (s->profiling) {
        MM_CUDA(cudaEventCreate(&e0));
        MM_CUDA(cudaEventCreate(&e1));
        s->ev.push_back(e0); s->ev.push_back(e1);
    }
    return s->L.nm == 5 ? launch_step_nm<5>(s, sc, e0, e1) : launch_step_nm<14>(s, sc, e0, e1);
}

int read_ctrl(mm_solver* s, Ctrl* h)
{
    MM_CUDA(cudaMemcpyAsync(h, s->ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, s->stream));
    MM_CUDA(cudaStreamSynchronize(s->stream));
    return MM_OK;
}

double bits2d(unsigned long long b) { double d; memcpy(&d, &b, 8); return d; }

template <int NM>
int set_state_impl(mm_solver* s, const double* src, int on_device, bool prim)
{
    const size_t nbytes = (size_t)NM * s->p.nx * s->p.ny * sizeof(double);
    const double* dsrc = src;
    if (!on_device) {   // stage through the idle state copy
        MM_CUDA(cudaMemcpyAsync(s->U[s->cur ^ 1], src, nbytes, cudaMemcpyHostToDevice, s->stream));
        dsrc = s->U[s->cur ^ 1];
    }
    dim3 grid((s->p.nx + 127) / 128, s->p.ny < 65535 ? s->p.ny : 65535);
    if (prim) k_pack<NM, true><<<grid, 128, 0, s->stream>>>(s->p, dsrc, s->U[s->cur], s->W[s->cur]);
    else k_pack<NM, false><<<grid, 128, 0, s->stream>>>(s->p, dsrc, s->U[s->cur], s->W[s->cur]);
    MM_LAUNCHED(s, "k_pack");
    if constexpr (NM == 14) {
        // the z-symmetric kernel variant leaves the z-odd planes alone: they are exact zeros in both copies
        // (the idle copy may hold the staged input)
        const int zodd[4] = {3, 6, 8, 12};
        for (int m : zodd) {
            MM_CUDA(cudaMemsetAsync(s->U[s->cur ^ 1] + (size_t)m * s->L.plane, 0, s->L.plane * sizeof(double), s->stream));
            MM_CUDA(cudaMemsetAsync(s->W[s->cur ^ 1] + (size_t)m * s->L.plane, 0, s->L.plane * sizeof(double), s->stream));
        }
    }
    // reset the clock and the accumulators (keeps the constant ghost part)
    MM_CUDA(cudaMemsetAsync(s->ctrl, 0, offsetof(Ctrl, ghost_rate), s->stream));
    MM_CUDA(cudaMemsetAsync(&s->ctrl->steps, 0, sizeof(Ctrl) - offsetof(Ctrl, steps), s->stream));
    s->slot = 0;
    s->hist_first = 0;
    StepCtl none = {0, 0.0, -1.0};
    int rc = launch_ghost<NM>(s, none, 0);
    if (rc) return rc;
    const long long n = (long long)s->p.nx * s->p.ny;
    int nb = (int)((n + kRateNT - 1) / kRateNT);
    if (nb > 148 * 8) nb = 148 * 8;
    k_rate<NM, kRateNT><<<nb, kRateNT, 0, s->stream>>>(s->p, s->U[s->cur], s->ctrl, 0);
    MM_LAUNCHED(s, "k_rate");
    s->has_state = 1;
    if constexpr (NM == 14) {        // fast-path precondition, checked on the device by k_rate / k_bc_table
        Ctrl h;
        if ((rc = read_ctrl(s, &h))) return rc;
        s->zsym = !h.znz && !h.bc_znz;
        // One pass of the step kernel with dt = 0 into the idle copy, for its CFL reduction alone: the rate of
        // the state is then the one the kernel's own tail computes -- the same instructions that produced it
        // in the run a checkpoint was taken from, so that set_state + set_clock resumes that run bit for bit
        // (k_rate's inlined copy of the wave-speed code may be fused differently by the compiler; W(U) from
        // k_pack is bit-identical by construction, see cons2prim14).  The pass's copy of the state is dropped.
        // ctrl->dt is 0 here (cleared above).  The pass must also be the INSTANTIATION whose tail produced the
        // rate in the original run: launch_pass picks the EXT variant for the point-implicit source by itself;
        // for the midpoint scheme the rate comes from a step's second pass, which has a base state, so this pass
        // is given one too (the state itself: B - 0 * div F = B).
        const double* base = s->time_scheme == MM_TIME_MIDPOINT ? s->U[s->cur] : nullptr;
        if ((rc = launch_pass(s, s->cur, s->cur ^ 1, base, 1.0, 1))) return rc;
        s->slot ^= 1;
    }
    return MM_OK;
}

template <int NM>
int get_state_impl(mm_solver* s, double* dst, int on_device, bool prim)
{
    const size_t nbytes = (size_t)NM * s->p.nx * s->p.ny * sizeof(double);
    double* ddst = on_device ? dst : s->U[s->cur ^ 1];
    dim3 grid((s->p.nx + 127) / 128, s->p.ny < 65535 ? s->p.ny : 65535);
    if (prim) k_unpack<NM, true><<<grid, 128, 0, s->stream>>>(s->p, s->U[s->cur], ddst);
    else k_unpack<NM, false><<<grid, 128, 0, s->stream>>>(s->p, s->U[s->cur], ddst);
    MM_LAUNCHED(s, "k_unpack");
    if (!on_device) {
        MM_CUDA(cudaMemcpyAsync(dst, ddst, nbytes, cudaMemcpyDeviceToHost, s->stream));
        if constexpr (NM == 14) {      // the idle copy served as staging: its z-odd planes are zeros again (see set_state_impl)
            const int zodd[4] = {3, 6, 8, 12};
            for (int m : zodd)
                MM_CUDA(cudaMemsetAsync(s->U[s->cur ^ 1] + (size_t)m * s->L.plane, 0, s->L.plane * sizeof(double), s->stream));
        }
    }
    MM_CUDA(cudaStreamSynchronize(s->stream));
    return MM_OK;
}

}  // namespace

extern "C" {

size_t mm_workspace_bytes(const mm_grid* grid)
{
    Layout L;
    return make_layout(grid, &L) ? L.total : 0;
}

int mm_create(mm_solver** out, const mm_grid* grid, const mm_gas* gas, const mm_collision* col,
              const mm_bc bcs[4], const mm_options* opt, void* d_workspace, size_t bytes)
{
    if (!out || !grid || !col || !bcs || !opt) return MM_EINVAL;
    if (gas && !(gas->R_gas > 0.0)) return MM_EINVAL;
    Layout L;
    if (!make_layout(grid, &L)) return MM_EINVAL;
    if (!(opt->sigma_lim > 0.0) || !(opt->ws_scale > 0.0)) return MM_EINVAL;
    if (opt->limiter < 0 || opt->limiter > 2 || opt->flux < 0 || opt->flux > 1) return MM_EINVAL;
    if (opt->source_scheme < 0 || opt->source_scheme > 1 || opt->time_scheme < 0 || opt->time_scheme > 1) return MM_EINVAL;
    if (opt->time_scheme == MM_TIME_MIDPOINT && opt->source_scheme != MM_SRC_EXPLICIT) return MM_EINVAL;
    if (col->model < 0 || col->model > 2) return MM_EINVAL;
    if (col->model == MM_TAU_CONST && !(col->tau > 0.0)) return MM_EINVAL;
    if (col->model == MM_TAU_KN && !(col->Kn > 0.0 && col->L_ref > 0.0 && col->rho_ref > 0.0)) return MM_EINVAL;
    const int ndim = grid->system == MM_SYS5_1D ? 1 : 2;
    for (int b = 0; b < 2 * ndim; ++b) {
        if (bcs[b].type < 0 || bcs[b].type > 2) return MM_EINVAL;
        if (bcs[b].type == MM_BC_DIRICHLET) {
            if (bcs[b].nbands < 0 || bcs[b].nbands > MM_MAX_BANDS) return MM_EINVAL;
            if (bcs[b].nbands > 0 && (!bcs[b].band_lo || !bcs[b].band_hi || !bcs[b].band_W)) return MM_EINVAL;
            if (bcs[b].band_state != MM_STATE_PRIMITIVE && bcs[b].band_state != MM_STATE_MAXWELLIAN) return MM_EINVAL;
        }
    }
    for (int d = 0; d < ndim; ++d)
        if ((bcs[2 * d].type == MM_BC_PERIODIC) != (bcs[2 * d + 1].type == MM_BC_PERIODIC)) return MM_EINVAL;
    if (!d_workspace || bytes < L.total || ((size_t)d_workspace & 255)) return MM_EWORKSPACE;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return cuda_fail(cudaErrorNoDevice, "mm_create (no CUDA device: this library has no CPU path)");

    mm_solver* s = new (std::nothrow) mm_solver();
    if (!s) return MM_EINVAL;
    s->grid = *grid; s->L = L;
    s->stream = (cudaStream_t)opt->stream;
    s->ws = (char*)d_workspace;
    s->ctrl = (Ctrl*)(s->ws + L.off_ctrl);
    s->bc = (BcTable*)(s->ws + L.off_bc);
    s->U[0] = (double*)(s->ws + L.off_u0);
    s->U[1] = (double*)(s->ws + L.off_u1);
    s->W[0] = L.nm == 14 ? (double*)(s->ws + L.off_w0) : nullptr;
    s->W[1] = L.nm == 14 ? (double*)(s->ws + L.off_w1) : nullptr;
    Params& p = s->p;
    p.sigma_lim = opt->sigma_lim; p.ws_scale = opt->ws_scale;
    p.dx = (grid->x1 - grid->x0) / grid->nx;
    p.dy = ndim == 2 ? (grid->y1 - grid->y0) / grid->ny : 1.0;
    p.x0 = grid->x0; p.y0 = ndim == 2 ? grid->y0 : 0.0;
    p.inv_dx = 1.0 / p.dx; p.inv_dy = 1.0 / p.dy;
    p.inv_tau_coef = col->model == MM_TAU_KN ? 1.0 / (col->Kn * col->L_ref * col->rho_ref) : 0.0;
    p.inv_tau_const = col->model == MM_TAU_CONST ? 1.0 / col->tau : 0.0;
    p.R_gas = gas ? gas->R_gas : 1.0;
    p.tau_model = col->model; p.limiter = opt->limiter;
    p.shared_limiter = opt->shared_limiter ? 1 : 0; p.flux = opt->flux;
    p.source_scheme = opt->source_scheme; s->time_scheme = opt->time_scheme;
    p.nx = grid->nx; p.ny = grid->ny; p.pitch = L.pitch; p.rows = L.rows;
    p.ab = (const double*)(s->ws + L.off_tab);
    p.set_constants();

    // boundary tables: copy, and mark which entries some ghost cell actually takes
    BcTable* hb = new (std::nothrow) BcTable();
    if (!hb) { delete s; return MM_EINVAL; }
    memset(hb, 0, sizeof *hb);
    const int nm = L.nm;
    for (int b = 0; b < 2 * ndim; ++b) {
        BcSide& sd = hb->side[b];
        sd.type = bcs[b].type;
        if (sd.type != MM_BC_DIRICHLET) continue;
        sd.nbands = bcs[b].nbands;
        sd.has_default = bcs[b].default_W ? 1 : 0;
        sd.maxwellian = bcs[b].band_state == MM_STATE_MAXWELLIAN;
        const int nw = sd.maxwellian ? 5 : nm;         // doubles per state as given (expanded by k_bc_table)
        for (int k = 0; k < sd.nbands; ++k) {
            sd.lo[k] = bcs[b].band_lo[k]; sd.hi[k] = bcs[b].band_hi[k];
            memcpy(sd.W[k], bcs[b].band_W + (size_t)k * nw, nw * sizeof(double));
        }
        if (sd.has_default) memcpy(sd.W[sd.nbands], bcs[b].default_W, nw * sizeof(double));
        const int n = b < 2 ? grid->ny : grid->nx;
        for (int pos = 0; pos < n; ++pos) {
            const double coord = b < 2 ? p.y0 + ((double)pos + 0.5) * p.dy : p.x0 + ((double)pos + 0.5) * p.dx;
            int k = sd.has_default ? sd.nbands : -1;
            for (int q = sd.nbands - 1; q >= 0; --q)
                if (coord >= sd.lo[q] && coord <= sd.hi[q]) k = q;
            if (k >= 0) sd.used |= 1u << k;
        }
    }
    cudaError_t e = cudaMemsetAsync(s->ws, 0, L.total, s->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(s->bc, hb, sizeof(BcTable), cudaMemcpyHostToDevice, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);   // hb is pageable: copy done before delete
    delete hb;
    if (e != cudaSuccess) { delete s; return cuda_fail(e, "mm_create workspace init"); }

    s->allow_fast = 1;
    if (nm == 14) {
        k_ab_table<<<AbTable::kIntervals, 2, 0, s->stream>>>((double*)(s->ws + L.off_tab));
        s->launches += 1;
        e = cudaFuncSetAttribute(k_step14_tm<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemGen);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_step14_tm<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemGen);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_step14_tm<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemZS);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_step14_tm<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemZS);
        if (e != cudaSuccess) { delete s; return cuda_fail(e, "cudaFuncSetAttribute(k_step14_tm)"); }
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        s->sms = sms;
        choose_decomposition(grid->nx, grid->ny, sms * kWarpsGen, &s->nstrips, &s->nchunks[0]);
        choose_decomposition(grid->nx, grid->ny, sms * kWarpsZS, &s->nstrips, &s->nchunks[1]);
        k_bc_table<14><<<4, kMaxBands + 1, 0, s->stream>>>(p, s->bc, s->ctrl, 4);
    } else {
        k_bc_table<5><<<2, kMaxBands + 1, 0, s->stream>>>(p, s->bc, s->ctrl, 2);
    }
    s->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) { delete s; return cuda_fail(e, "k_bc_table"); }
    *out = s;
    return MM_OK;
}

int mm_set_state(mm_solver* s, const double* U, int on_device)
{
    if (!s || !U) return MM_EINVAL;
    return s->L.nm == 5 ? set_state_impl<5>(s, U, on_device, false) : set_state_impl<14>(s, U, on_device, false);
}

int mm_set_state_prim(mm_solver* s, const double* W, int on_device)
{
    if (!s || !W) return MM_EINVAL;
    return s->L.nm == 5 ? set_state_impl<5>(s, W, on_device, true) : set_state_impl<14>(s, W, on_device, true);
}

int mm_get_state(mm_solver* s, double* U, int on_device)
{
    if (!s || !U || !s->has_state) return MM_EINVAL;
    return s->L.nm == 5 ? get_state_impl<5>(s, U, on_device, false) : get_state_impl<14>(s, U, on_device, false);
}

int mm_get_state_prim(mm_solver* s, double* W, int on_device)
{
    if (!s || !W || !s->has_state) return MM_EINVAL;
    return s->L.nm == 5 ? get_state_impl<5>(s, W, on_device, true) : get_state_impl<14>(s, W, on_device, true);
}

int mm_step(mm_solver* s, int n, double cfl)
{
    if (!s || n < 0 || !(cfl > 0.0) || !s->has_state) return MM_EINVAL;
    StepCtl sc = {1, cfl, -1.0};
    for (int k = 0; k < n; ++k) {
        int rc = launch_step(s, sc);
        if (rc) return rc;
    }
    return MM_OK;
}

int mm_step_fixed_dt(mm_solver* s, int n, double dt)
{
    if (!s || n < 0 || !(dt > 0.0) || !s->has_state) return MM_EINVAL;
    StepCtl sc = {0, dt, -1.0};
    for (int k = 0; k < n; ++k) {
        int rc = launch_step(s, sc);
        if (rc) return rc;
    }
    return MM_OK;
}

int mm_advance_to(mm_solver* s, double t_end, double cfl, int max_steps)
{
    if (!s || !(cfl > 0.0) || !(t_end >= 0.0) || !s->has_state) return MM_EINVAL;
    Ctrl h;
    int rc = read_ctrl(s, &h);
    if (rc) return rc;
    const long long first = h.steps;
    StepCtl sc = {1, cfl, t_end};
    while (h.t < t_end && !h.failed) {
        long long left = max_steps > 0 ? max_steps - (h.steps - first) : (1ll << 40);
        if (left <= 0) break;
        // enqueue about as many steps as the current dt suggests; steps past t_end only copy
        double rate = fmax(bits2d(h.rate_bits[s->slot]), h.ghost_rate);
        double est = rate > 0.0 ? (t_end - h.t) * rate / cfl : 1.0;
        long long batch = est < 1.0 ? 1 : (est > 256.0 ? 256 : (long long)est + 1);
        if (batch > left) batch = left;
        for (long long k = 0; k < batch; ++k)
            if ((rc = launch_step(s, sc))) return rc;
        if ((rc = read_ctrl(s, &h))) return rc;
    }
    return h.failed ? MM_ENONFINITE : MM_OK;
}

int mm_get_info(mm_solver* s, double* t, long long* steps, double* last_dt, double* max_speed)
{
    if (!s) return MM_EINVAL;
    Ctrl h;
    int rc = read_ctrl(s, &h);
    if (rc) return rc;
    if (t) *t = h.t;
    if (steps) *steps = h.steps;
    if (last_dt) *last_dt = h.last_dt;
    if (max_speed) *max_speed = fmax(bits2d(h.speed_bits[s->slot]), h.ghost_speed);
    return (h.failed || h.bc_bad || h.bad[s->slot]) ? MM_ENONFINITE : MM_OK;
}

int mm_cfl_dt(mm_solver* s, double cfl, double* dt)
{
    if (!s || !dt || !(cfl > 0.0) || !s->has_state) return MM_EINVAL;
    Ctrl h;
    int rc = read_ctrl(s, &h);
    if (rc) return rc;
    double rate = fmax(bits2d(h.rate_bits[s->slot]), h.ghost_rate);
    if (h.failed || h.bc_bad || h.bad[s->slot] || !(rate > 0.0)) return MM_ENONFINITE;
    *dt = cfl / rate;
    return MM_OK;
}

int mm_get_dt_history(mm_solver* s, long long first_step, int n, double* dt)
{
    if (!s || !dt || n < 0 || first_step < 0) return MM_EINVAL;
    if (n == 0) return MM_OK;
    Ctrl h;
    int rc = read_ctrl(s, &h);
    if (rc) return rc;
    if (first_step < s->hist_first) return MM_EINVAL;                                      // before this solver's own steps
    if (first_step + n > h.steps || h.steps - first_step > kDtHistory) return MM_EINVAL;   // not taken yet / overwritten
    const double* hist = (const double*)(s->ws + s->L.off_hist);
    for (int k = 0; k < n;) {                      // the ring wraps at most once inside the range
        const long long pos = (first_step + k) & (kDtHistory - 1);
        const int run = (int)((long long)(n - k) < kDtHistory - pos ? (n - k) : kDtHistory - pos);
        MM_CUDA(cudaMemcpyAsync(dt + k, hist + pos, (size_t)run * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        k += run;
    }
    MM_CUDA(cudaStreamSynchronize(s->stream));
    return MM_OK;
}

int mm_set_clock(mm_solver* s, double t, long long steps)
{
    if (!s || !s->has_state || !(t >= 0.0) || steps < 0) return MM_EINVAL;
    MM_CUDA(cudaMemcpyAsync(&s->ctrl->t, &t, sizeof t, cudaMemcpyHostToDevice, s->stream));
    MM_CUDA(cudaMemcpyAsync(&s->ctrl->steps, &steps, sizeof steps, cudaMemcpyHostToDevice, s->stream));
    MM_CUDA(cudaStreamSynchronize(s->stream));     // t and steps are stack variables
    s->hist_first = steps;                         // steps before the restored counter were not taken here
    return MM_OK;
}

long long mm_launch_count(const mm_solver* s) { return s ? s->launches : 0; }

int mm_decomposition(int nx, int ny, int zsym, int sms, int* nstrips, int* nchunks, int* warps_per_sm)
{
    if (nx < 1 || ny < 1 || sms < 1 || !nstrips || !nchunks || !warps_per_sm) return MM_EINVAL;
    const int nw = zsym ? kWarpsZS : kWarpsGen;
    choose_decomposition(nx, ny, sms * nw, nstrips, nchunks);
    *warps_per_sm = nw;
    return MM_OK;
}

int mm_set_fast_path(mm_solver* s, int allow)
{
    if (!s) return MM_EINVAL;
    s->allow_fast = allow ? 1 : 0;
    return MM_OK;
}

int mm_fast_path_active(const mm_solver* s) { return s ? (s->zsym && s->allow_fast && s->L.nm == 14) : 0; }

int mm_profile_begin(mm_solver* s)
{
    if (!s) return MM_EINVAL;
    for (cudaEvent_t e : s->ev) cudaEventDestroy(e);
    s->ev.clear();
    s->profiling = true;
    return MM_OK;
}

int mm_profile_end(mm_solver* s, double* step_kernel_ms, long long* launches)
{
    if (!s || !s->profiling) return MM_EINVAL;
    s->profiling = false;
    MM_CUDA(cudaStreamSynchronize(s->stream));
    double total = 0.0;
    for (size_t k = 0; k + 1 < s->ev.size(); k += 2) {
        float ms = 0.f;
        MM_CUDA(cudaEventElapsedTime(&ms, s->ev[k], s->ev[k + 1]));
        total += ms;
    }
    if (step_kernel_ms) *step_kernel_ms = total;
    if (launches) *launches = (long long)(s->ev.size() / 2);
    for (cudaEvent_t e : s->ev) cudaEventDestroy(e);
    s->ev.clear();
    return MM_OK;
}

// ---------------------------------------------------------------- batched 1-D 5-moment tubes
struct mm_batch5 {
    int nx, ntubes;
    Params p;
    cudaStream_t stream;
    char* ws;
    TubeCtl* ctl;
    double *sigma_lim, *inv_tau_coef, *U[2];
    size_t state_bytes;
    int cur, slot, has_state;
    long long launches;
};

namespace {
constexpr int kNTB = 128;
struct BLayout { size_t off_ctl, off_sig, off_itc, off_u0, off_u1, state_bytes, total; };
bool batch_layout(int nx, int ntubes, BLayout* L)
{
    if (nx < 1 || ntubes < 1 || ntubes > 65535) return false;
    L->state_bytes = align_up((size_t)ntubes * 5 * nx * sizeof(double), 256);
    L->off_ctl = 0;
    L->off_sig = align_up((size_t)ntubes * sizeof(TubeCtl), 256);
    L->off_itc = L->off_sig + align_up((size_t)ntubes * sizeof(double), 256);
    L->off_u0 = L->off_itc + align_up((size_t)ntubes * sizeof(double), 256);
    L->off_u1 = L->off_u0 + L->state_bytes;
    L->total = L->off_u1 + L->state_bytes;
    return true;
}
int batch_step(mm_batch5* b, const StepCtl& sc)
{
    k_batch5_finalize<<<(b->ntubes + 127) / 128, 128, 0, b->stream>>>(b->ntubes, b->ctl, b->slot, sc);
    dim3 grid((b->nx + kNTB - 2) / (kNTB - 1), b->ntubes);       // kNTB - 1 cells per block (mm_batch5.cuh)
    k_batch5_step<kNTB><<<grid, kNTB, 0, b->stream>>>(b->p, b->sigma_lim, b->inv_tau_coef, b->U[b->cur],
                                                     b->U[b->cur ^ 1], b->ctl, b->slot ^ 1);
    b->launches += 2;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "k_batch5_step");
    b->cur ^= 1; b->slot ^= 1;
    return MM_OK;
}
int batch_read_ctl(mm_batch5* b, std::vector<TubeCtl>& h)
{
    h.resize(b->ntubes);
    MM_CUDA(cudaMemcpyAsync(h.data(), b->ctl, (size_t)b->ntubes * sizeof(TubeCtl), cudaMemcpyDeviceToHost, b->stream));
    MM_CUDA(cudaStreamSynchronize(b->stream));
    return MM_OK;
}
}  // namespace

size_t mm_batch5_workspace_bytes(int nx, int ntubes)
{
    BLayout L;
    return batch_layout(nx, ntubes, &L) ? L.total : 0;
}

int mm_batch5_create(mm_batch5** out, int nx, int ntubes, double x0, double x1, const double* sigma_lim,
                     const double* Kn, double L_ref, double rho_ref, double ws_scale, int limiter,
                     int shared_limiter, int flux, void* stream, void* d_workspace, size_t bytes)
{
    if (!out || !sigma_lim || !Kn || !(x1 > x0) || !(ws_scale > 0.0) || !(L_ref > 0.0) || !(rho_ref > 0.0)) return MM_EINVAL;
    if (limiter < 0 || limiter > 2 || flux < 0 || flux > 1) return MM_EINVAL;
    BLayout L;
    if (!batch_layout(nx, ntubes, &L)) return MM_EINVAL;
    for (int j = 0; j < ntubes; ++j) if (!(sigma_lim[j] > 0.0)) return MM_EINVAL;
    if (!d_workspace || bytes < L.total || ((size_t)d_workspace & 255)) return MM_EWORKSPACE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return cuda_fail(cudaErrorNoDevice, "mm_batch5_create (no CUDA device: this library has no CPU path)");
    mm_batch5* b = new (std::nothrow) mm_batch5();
    if (!b) return MM_EINVAL;
    b->nx = nx; b->ntubes = ntubes; b->stream = (cudaStream_t)stream; b->ws = (char*)d_workspace;
    b->ctl = (TubeCtl*)(b->ws + L.off_ctl);
    b->sigma_lim = (double*)(b->ws + L.off_sig); b->inv_tau_coef = (double*)(b->ws + L.off_itc);
    b->U[0] = (double*)(b->ws + L.off_u0); b->U[1] = (double*)(b->ws + L.off_u1);
    b->state_bytes = L.state_bytes;
    Params& p = b->p;
    memset(&p, 0, sizeof p);
    p.ws_scale = ws_scale; p.dx = (x1 - x0) / nx; p.dy = 1.0; p.x0 = x0;
    p.inv_dx = 1.0 / p.dx; p.inv_dy = 1.0;
    p.limiter = limiter; p.shared_limiter = shared_limiter ? 1 : 0; p.flux = flux;
    p.nx = nx; p.ny = 1;
    p.set_constants();
    std::vector<double> itc(ntubes);
    for (int j = 0; j < ntubes; ++j) itc[j] = Kn[j] > 0.0 ? 1.0 / (Kn[j] * L_ref * rho_ref) : 0.0;   // <= 0: collisionless
    cudaError_t e = cudaMemsetAsync(b->ws, 0, L.off_u0, b->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(b->sigma_lim, sigma_lim, ntubes * sizeof(double), cudaMemcpyHostToDevice, b->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(b->inv_tau_coef, itc.data(), ntubes * sizeof(double), cudaMemcpyHostToDevice, b->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(b->stream);
    if (e != cudaSuccess) { delete b; return cuda_fail(e, "mm_batch5_create"); }
    *out = b;
    return MM_OK;
}

int mm_batch5_set_state_prim(mm_batch5* b, const double* W, int per_tube, int on_device)
{
    if (!b || !W) return MM_EINVAL;
    const size_t nbytes = (size_t)(per_tube ? b->ntubes : 1) * 5 * b->nx * sizeof(double);
    const double* src = W;
    if (!on_device) {
        MM_CUDA(cudaMemcpyAsync(b->U[b->cur ^ 1], W, nbytes, cudaMemcpyHostToDevice, b->stream));
        src = b->U[b->cur ^ 1];
    }
    dim3 grid((b->nx + 127) / 128, b->ntubes);
    k_batch5_pack<<<grid, 128, 0, b->stream>>>(b->nx, b->ntubes, per_tube ? 1 : 0, src, b->U[b->cur]);
    MM_CUDA(cudaGetLastError());
    MM_CUDA(cudaMemsetAsync(b->ctl, 0, (size_t)b->ntubes * sizeof(TubeCtl), b->stream));
    b->slot = 0;
    dim3 g2((b->nx + kNTB - 1) / kNTB, b->ntubes);
    k_batch5_rate<kNTB><<<g2, kNTB, 0, b->stream>>>(b->p, b->sigma_lim, b->inv_tau_coef, b->U[b->cur], b->ctl);
    b->launches += 2;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "mm_batch5_set_state_prim");
    b->has_state = 1;
    return MM_OK;
}

int mm_batch5_step(mm_batch5* b, int n, double cfl)
{
    if (!b || n < 0 || !(cfl > 0.0) || !b->has_state) return MM_EINVAL;
    StepCtl sc = {1, cfl, -1.0};
    for (int k = 0; k < n; ++k) { int rc = batch_step(b, sc); if (rc) return rc; }
    return MM_OK;
}

int mm_batch5_step_fixed_dt(mm_batch5* b, int n, double dt)
{
    if (!b || n < 0 || !(dt > 0.0) || !b->has_state) return MM_EINVAL;
    StepCtl sc = {0, dt, -1.0};
    for (int k = 0; k < n; ++k) { int rc = batch_step(b, sc); if (rc) return rc; }
    return MM_OK;
}

int mm_batch5_advance_to(mm_batch5* b, double t_end, double cfl, long long max_steps)
{
    if (!b || !(cfl > 0.0) || !(t_end >= 0.0) || !b->has_state) return MM_EINVAL;
    StepCtl sc = {1, cfl, t_end};
    std::vector<TubeCtl> h;
    long long done = 0;
    for (;;) {
        int rc = batch_read_ctl(b, h);
        if (rc) return rc;
        double need = 0.0;                      // steps the slowest unfinished tube still needs, estimated
        for (const TubeCtl& c : h) {
            if (c.failed || c.t >= t_end) continue;
            const double rate = bits2d(c.rate_bits[b->slot]);
            const double est = rate > 0.0 ? (t_end - c.t) * rate / cfl : 1.0;
            if (est > need) need = est;
        }
        if (need <= 0.0 || (max_steps > 0 && done >= max_steps)) break;
        long long batch = need < 1.0 ? 1 : (need > 512.0 ? 512 : (long long)need + 1);
        if (max_steps > 0 && batch > max_steps - done) batch = max_steps - done;
        for (long long k = 0; k < batch; ++k) if ((rc = batch_step(b, sc))) return rc;
        done += batch;
    }
    return MM_OK;
}

int mm_batch5_get_state(mm_batch5* b, double* U, int on_device)
{
    if (!b || !U || !b->has_state) return MM_EINVAL;
    const size_t nbytes = (size_t)b->ntubes * 5 * b->nx * sizeof(double);
    MM_CUDA(cudaMemcpyAsync(U, b->U[b->cur], nbytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, b->stream));
    MM_CUDA(cudaStreamSynchronize(b->stream));
    return MM_OK;
}

int mm_batch5_get_info(mm_batch5* b, double* t, long long* steps, int* failed)
{
    if (!b) return MM_EINVAL;
    std::vector<TubeCtl> h;
    int rc = batch_read_ctl(b, h);
    if (rc) return rc;
    int any = 0;
    for (int j = 0; j < b->ntubes; ++j) {
        const int f = h[j].failed || h[j].bad[b->slot];
        if (t) t[j] = h[j].t;
        if (steps) steps[j] = h[j].steps;
        if (failed) failed[j] = f;
        any |= f;
    }
    return any ? MM_ENONFINITE : MM_OK;
}

long long mm_batch5_launch_count(const mm_batch5* b) { return b ? b->launches : 0; }
void mm_batch5_destroy(mm_batch5* b) { delete b; }

void mm_destroy(mm_solver* s)
{
    if (!s) return;
    for (cudaEvent_t e : s->ev) cudaEventDestroy(e);
    delete s;
}

const char* mm_strerror(int status)
{
    switch (status) {
    case MM_OK: return "ok";
    case MM_EINVAL: return "invalid argument";
    case MM_EWORKSPACE: return "workspace missing, too small or not 256-byte aligned";
    case MM_ECUDA: return g_cuda_msg[0] ? g_cuda_msg : "CUDA error";
    case MM_ENONFINITE: return "CFL reduction met rho <= 0, P <= 0 or a non-finite wave speed";
    case MM_ETOOLARGE: return "problem larger than the library's built-in scratch: mm_static5_run takes at most "
                              "MM_STATIC5_MAX_NX = 8192 cells (use mm_create with a workspace of your own beyond that)";
    default: return "unknown status";
    }
}

}  // extern "C"

// ---------------------------------------------------------------- run without a caller workspace
// mm_static5_run (include/mm.h) serves callers that can hand over their input and output arrays but no
// device workspace: callbacks living inside a host application that owns all device memory, loops that
// must not hit the device-wide synchronisation of a runtime allocation, drivers without a CUDA runtime of
// their own.  The scratch of the 5-moment step -- everything mm_workspace_bytes() would have asked the
// caller for -- is this one array in the library image instead: 4 MiB on every GPU that loads libmm.so,
// until the process exits.
namespace {

static __device__ __align__(256) unsigned char g_static5_scratch[MM_STATIC5_SCRATCH_BYTES];

// In host code `g_static5_scratch` is only the handle the runtime knows the array by, not an address a
// kernel could use.  The usable device address differs per device; it is looked up once per device, with
// that device current, and kept here.
constexpr int kStatic5MaxDevices = 64;
void* g_static5_addr[kStatic5MaxDevices];
std::mutex g_static5_mu;        // one call at a time: all calls on a device share the array

int static5_scratch_address(void** out)
{
    int dev = -1;
    MM_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStatic5MaxDevices) return MM_EINVAL;
    if (!g_static5_addr[dev]) {
        void* p = nullptr;
        MM_CUDA(cudaGetSymbolAddress(&p, g_static5_scratch));
        if (!p) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_static5_scratch)");
        g_static5_addr[dev] = p;
    }
    *out = g_static5_addr[dev];
    return MM_OK;
}

}  // namespace

extern "C" int mm_static5_run(int nx, double x0, double x1, const mm_collision* collision, const mm_bc* bcs,
                              const mm_options* options, const double* W0, int n, double cfl, double dt,
                              double* U, int on_device, double* t_end)
{
    if (!collision || !options || !W0 || !U || nx < 1 || n < 0) return MM_EINVAL;
    if (!(dt > 0.0) && !(cfl > 0.0)) return MM_EINVAL;
    if (nx > MM_STATIC5_MAX_NX) return MM_ETOOLARGE;            // before any CUDA call
    const mm_grid g = {MM_SYS5_1D, nx, 1, x0, x1, 0.0, 1.0};
    Layout L;
    if (!make_layout(&g, &L)) return MM_EINVAL;
    if (L.total > (size_t)MM_STATIC5_SCRATCH_BYTES) return MM_ETOOLARGE;
    mm_bc sides[4];
    memset(sides, 0, sizeof sides);                              // MM_BC_TRANSMISSIVE
    if (bcs) { sides[0] = bcs[0]; sides[1] = bcs[1]; }

    std::lock_guard<std::mutex> lock(g_static5_mu);
    void* scratch = nullptr;
    int rc = static5_scratch_address(&scratch);                  // first call on this device: module load + lookup
    if (rc) return rc;
    // mm_create zero-fills the L.total bytes this problem uses (the array still holds the previous call's
    // control block, tables and states) and rebuilds the boundary table; the solver object is host memory.
    mm_solver* s = nullptr;
    if ((rc = mm_create(&s, &g, nullptr, collision, sides, options, scratch, MM_STATIC5_SCRATCH_BYTES))) return rc;
    rc = mm_set_state_prim(s, W0, on_device);
    if (!rc) rc = dt > 0.0 ? mm_step_fixed_dt(s, n, dt) : mm_step(s, n, cfl);
    if (!rc) rc = mm_get_state(s, U, on_device);
    if (!rc) rc = mm_get_info(s, t_end, nullptr, nullptr, nullptr);
    // whatever happened, nothing of this call may still be running on the array when the lock is released
    const cudaError_t e = cudaStreamSynchronize(s->stream);
    mm_destroy(s);
    if (!rc && e != cudaSuccess) rc = cuda_fail(e, "mm_static5_run: cudaStreamSynchronize");
    return rc;
}
