// fvnl.cu -- C-ABI library of the B200-native finite-volume step of arXiv 1311.3004 (include/fvnl.h).
//
// Host side: context, argument checks, launch sequence.  All arithmetic of the path runs in the kernels: the
// warp-specialised one-pass step kernel of fvnl_ws.cuh (default), the single-role one-pass kernel of fvnl_fused.cuh and the
// three-pass kernels of fvnl_unfused.cuh (opt-in comparison paths), the clock / pre-pass / boundary kernels below; there is
// no CPU fallback.
// Build: paper_1311_3004_b200/build.py (nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo).
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/fvnl.h"
#include "fvnl_ws.cuh"
#include "fvnl_small.cuh"

using namespace fvnl;

// ---------------------------------------------------------------------------------------------------------------
// Clock kernels (one thread).  PAPER.md:275-279, readings A7, A8.  The end of a step (M_n, nu_n, t += dt and
// the next dt) is NOT a kernel: the block of the step kernel that finishes last does it (step_tail, fvnl_fused.cuh).

// fvnl_set_state: sticky flags and the lagged maximum are reset, t and the step counter stay.
__global__ void k_clock_reset(Clock* c) {
    c->flags = 0;
    c->Mprev = 0.0;
    c->sx_bits = c->sy_bits = 0ull;
    c->ticket = 0u;
}

// fvnl_set_clock.
__global__ void k_clock_set(Clock* c, double t, double M) {
    c->t = t;
    c->Mprev = M;
    c->sx_bits = c->sy_bits = 0ull;
    c->ticket = 0u;
}

// Start of a fvnl_step call.  from_prepass: M_{n-1} is what k_prepass has just left in sx_bits / sy_bits.
// mode 0: value = dt; mode 1: value = nu_W, dt = nu_W / (c0 M_prev).
__global__ void k_clock_begin(Grid g, Clock* c, double value, int mode, int from_prepass) {
    if (from_prepass) {
        const double sx = __longlong_as_double((long long)c->sx_bits), sy = __longlong_as_double((long long)c->sy_bits);
        c->Mprev = fmax(__ddiv_rn(sx, g.dx), __ddiv_rn(sy, g.dy));
    }
    clock_set_dt(g, c, value, mode, c->Mprev);
}

// End of a step for the three-pass comparison path (its kernels have no tail).
__global__ void k_clock_end(Grid g, Clock* c, double value, int mode, int more) { clock_advance(g, c, value, mode, more); }

// The speed that enters M at one interface: max_p |s^p| = |v| + a of (32)-(34), which depends on the
// density and the NORMAL velocity of the two cells only (z = q2/q1 for an x-interface, q3/q1 for a y-interface).
__device__ __forceinline__ double iface_speed(double q1L, double zL, double q1R, double zR, double b2, double omb2, int& min_dhi) {
    const double Zb1 = 0.5 * (q1L + q1R), Zb2 = 0.5 * (zL + zR);
    const double v = Zb2 * rcp_o1(Zb1);
    const double disc = fma(v, fma(-2.0, Zb2, v), fma(b2, Zb1, omb2));
    min_dhi = min(min_dhi, hi_word(disc));
    return fabs(v) + disc * rsqrt_o1(disc);
}

// O7 pre-pass: M of the current state = max |s|/h over the x-interfaces of G_x(Q) and the y-interfaces of G_y(Q) that
// touch an interior cell (first step of CFL mode).  A read-only pass at HBM rate: every warp marches down a chunk of
// PRE_ROWS rows over 32 consecutive columns (31 new ones + the left neighbour, handed over by shuffle -- no shared memory,
// no barrier), the row below is carried in registers; analytic ghost cells come from k_sources' buffer.
// grid = (ceil((nx + 1) / 124), ceil(ny / PRE_ROWS)), block = 128.
constexpr int PRE_ROWS = 64;
template <class T>
__global__ void __launch_bounds__(128) k_prepass(Grid g, Clock* clk, const T* __restrict__ q1, const T* __restrict__ q2,
                                                 const T* __restrict__ q3) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int i_raw = ((int)blockIdx.x * 4 + warp) * 31 + lane - 1;           // column on the ghost-extended mesh, from -1
    const int i = min(i_raw, g.nx);                                           // (lanes beyond the mesh idle on column nx)
    const int j0 = (int)blockIdx.y * PRE_ROWS, j1 = min(j0 + PRE_ROWS, g.ny);
    const int rlast = j1 == g.ny ? g.ny : j1 - 1;                             // the top chunk also owns interface ny - 1/2 + 1
    const bool x_if = lane >= 1 && i_raw <= g.nx;                             // x-interface i - 1/2, i = 0 .. nx
    const bool y_col = lane >= 1 && i_raw < g.nx;                             // y-interfaces of an interior column
    const ColMap cm = map_column(g, i);
    const double* src = src_buffer(g, clk->steps);
    const double b2 = 2.0 * (g.beta - 1.0), omb2 = 1.0 - b2;
    double sx = 0.0, sy = 0.0, below_q1 = 1.0, below_z3 = 0.0;
    int mq = 0x7fffffff, md = 0x7fffffff;
#pragma unroll 4
    for (int r = j0 - 1; r <= rlast; ++r) {
        const Q3 c = load_mapped(g, src, cm, i, r, q1, q2, q3);
        mq = min(mq, hi_word(c.q1));
        const double rc = rcp_o1(c.q1), z2 = c.q2 * rc, z3 = c.q3 * rc;
        const double left_q1 = __shfl_up_sync(0xffffffffu, c.q1, 1), left_z2 = __shfl_up_sync(0xffffffffu, z2, 1);
        if (x_if && r >= j0 && r < g.ny) sx = fmax(sx, iface_speed(left_q1, left_z2, c.q1, z2, b2, omb2, md));
        if (y_col && r >= j0) sy = fmax(sy, iface_speed(below_q1, below_z3, c.q1, z3, b2, omb2, md));
        below_q1 = c.q1; below_z3 = z3;
    }
    int flags = 0;
    if (i_raw <= g.nx && mq <= 0) flags |= F_ENONPOS;
    if (md < 0) flags |= F_ENONREAL;
    block_max_to(&clk->sx_bits, sx);
    __syncthreads();
    block_max_to(&clk->sy_bits, sy);
    block_flags_to(&clk->flags, flags);
}

// Boundary / source-injection kernel: the analytic ghost cells (41), (43a-d), piston of every SOURCE side at t_n
// (readings A11, A13, A14, A16), three layers deep, into Grid::src.  One thread per record.
__global__ void __launch_bounds__(128) k_sources(Grid g, const Clock* clk) {
    const size_t n = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (n < src_off(g.nx, g.ny, 4) / 3) source_record(g, clk->t, n, src_buffer(g, clk->steps));
}

__global__ void k_fill(double* p, size_t n, double v) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = v;
}

// fp32 contexts: conversion between the standard fp64 state q and the stored planes (rho' = q1 - 1, q2, q3) in fp32.
__global__ void k_to_f32(const double* __restrict__ q1, const double* __restrict__ q2, const double* __restrict__ q3,
                         float* __restrict__ r, float* __restrict__ m2, float* __restrict__ m3, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        r[i] = (float)(q1[i] - 1.0); m2[i] = (float)q2[i]; m3[i] = (float)q3[i];
    }
}
__global__ void k_from_f32(const float* __restrict__ r, const float* __restrict__ m2, const float* __restrict__ m3,
                           double* __restrict__ q1, double* __restrict__ q2, double* __restrict__ q3, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        q1[i] = 1.0 + (double)r[i]; q2[i] = (double)m2[i]; q3[i] = (double)m3[i];
    }
}

// fvnl_shift: the domain moves k cells in +x (second stage of PAPER.md:287).  Q_new(i, j) = Q_old(i + k, j); the k columns
// that enter on the right are the x-hi ghost cells of the old state by the x-hi rule at the current time: zero-order
// extrapolation, or the analytic cell at its own centre (inside the aperture).  One thread per cell.
template <class T>
__global__ void __launch_bounds__(256) k_shift(Grid g, const Clock* clk, int k, const T* __restrict__ a1, const T* __restrict__ a2,
                                               const T* __restrict__ a3, T* __restrict__ o1, T* __restrict__ o2,
                                               T* __restrict__ o3) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= g.nx) return;
    const size_t o = (size_t)j * g.nx + i;
    const int io = i + k;
    if (io < g.nx) { o1[o] = a1[o + k]; o2[o] = a2[o + k]; o3[o] = a3[o + k]; return; }
    const size_t e = (size_t)j * g.nx + g.nx - 1;
    T c1 = a1[e], c2 = a2[e], c3 = a3[e];
    Q3 s;
    if (g.side[SIDE_XHI].kind == BC_SOURCE && source_at(g, SIDE_XHI, io, j, clk->t, s)) {
        c1 = dens_var<T>(s.q1); c2 = T(s.q2); c3 = T(s.q3);
    }
    o1[o] = c1; o2[o] = c2; o3[o] = c3;
}

// ---------------------------------------------------------------------------------------------------------------
struct fvnl_ctx {
    Grid g;
    int device;
    cudaStream_t stream;
    size_t n;                   // nx*ny
    void* ws;                   // workspace base
    bool own_ws;
    Clock* clk;                 // device clock
    double* src;                // analytic ghost cells of SOURCE sides, two buffers (src_buffer)
    int prec;                   // 64 or 32
    size_t elem;                // bytes of a state value
    char* buf[2][3];            // two state buffers (ping-pong) of `prec`-bit planes; cur = index of the current state
    int cur;
    double* star[3];            // unfused path only: Q* on the y-extended mesh, allocated on first use
    Clock* host_clk;            // pinned
    Clock snap;                 // last read-back
    bool have_state;
    bool need_prepass;
    int kernel;                 // FVNL_KERNEL_*
    int rows_per_block;         // fused kernel: rows per chunk (0 = automatic)
    int variant;                // fused kernel: launch variant
    int small;                  // FVNL_OPT_SMALL_GRID: 1 = grids of at most SMALL_MAX_CELLS cells run all steps of a call in one
                                // cluster launch (k_steps_cluster), 0 = never
    int small_cluster;          // CTAs per cluster the device accepts for it (0 = not probed yet, -1 = unavailable)
    long launches;
    // CUDA graph of two consecutive steps (state A -> B -> A), for grids so small that launches dominate
    cudaStream_t gstream;       // capture stream (never executes anything)
    cudaGraphExec_t gexec;
    bool gvalid;
    double gvalue;
    int gmode, gcur, gvariant, grows;
    // opt-in per-kernel timing (FVNL_OPT_KERNEL_TIMING): event pairs around the sweep kernels, resolved on demand
    bool timing;
    struct Span { int id; cudaEvent_t a, b; };
    std::vector<Span>* spans;
    double span_ms[FVNL_TIMED_KINDS];
    long span_n[FVNL_TIMED_KINDS];
};

static const size_t MAX_SPANS = 1 << 16;
static const int N_FUSED_VARIANTS = 2;      // 0: k_step_ws (default), 1: k_step_fused
static const int DEFAULT_VARIANT = 0;
static const int FUSED_BX = 128, FUSED_MINB = 3;     // k_step_fused: block width, blocks per SM of its register budget

// Event pair around one kernel launch (timing on only).
struct SpanGuard {
    fvnl_ctx* c;
    cudaEvent_t b;
    SpanGuard(fvnl_ctx* c_, int id) : c(c_), b(nullptr) {
        if (!c->timing || c->spans->size() >= MAX_SPANS) return;
        cudaEvent_t a;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { (void)cudaGetLastError(); b = nullptr; return; }
        cudaEventRecord(a, c->stream);
        c->spans->push_back({id, a, b});
    }
    ~SpanGuard() { if (b) cudaEventRecord(b, c->stream); }
};

static void resolve_spans(fvnl_ctx* c) {
    if (!c->spans) return;
    for (auto& s : *c->spans) {
        float ms = 0.f;
        if (cudaEventSynchronize(s.b) == cudaSuccess && cudaEventElapsedTime(&ms, s.a, s.b) == cudaSuccess) {
            c->span_ms[s.id] += ms;
            c->span_n[s.id] += 1;
        }
        cudaEventDestroy(s.a);
        cudaEventDestroy(s.b);
    }
    (void)cudaGetLastError();
    c->spans->clear();
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static const size_t CLOCK_BYTES = 256;

extern "C" size_t fvnl_workspace_bytes(int nx, int ny, int precision) {
    if (nx < 4 || ny < 4 || (precision != 64 && precision != 32)) return 0;
    const size_t plane = align_up((size_t)nx * ny * (precision / 8), 256);
    return CLOCK_BYTES + 6 * plane + align_up(2 * src_stride(nx, ny) * sizeof(double), 256);
}

#define CK(call)                                         \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) { (void)cudaGetLastError(); return FVNL_ECUDA; } \
    } while (0)

extern "C" int fvnl_create(fvnl_ctx** out, int nx, int ny, double dx, double dy, const fvnl_medium* m, int precision,
                           void* cuda_stream, void* workspace, size_t workspace_bytes) {
    if (!out) return FVNL_EARG;
    *out = nullptr;
    if (nx < 4 || ny < 4 || !(dx > 0) || !(dy > 0) || !m || !(m->c0 > 0) || !(m->rho0 > 0) || !(m->beta >= 1) ||
        !(m->delta >= 0) || (precision != 64 && precision != 32))
        return FVNL_EARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { (void)cudaGetLastError(); return FVNL_ECUDA; }
    fvnl_ctx* c = new (std::nothrow) fvnl_ctx();
    if (!c) return FVNL_EALLOC;
    std::memset(c, 0, sizeof(*c));
    c->spans = new (std::nothrow) std::vector<fvnl_ctx::Span>();
    if (!c->spans) { delete c; return FVNL_EALLOC; }
    if (cudaGetDevice(&c->device) != cudaSuccess) { delete c; return FVNL_ECUDA; }
    c->g.nx = nx; c->g.ny = ny; c->g.dx = dx; c->g.dy = dy;
    c->g.c0 = m->c0; c->g.beta = m->beta; c->g.delta = m->delta;
    for (int s = 0; s < 4; ++s) c->g.side[s].kind = BC_EXTRAP;
    c->stream = (cudaStream_t)cuda_stream;
    c->n = (size_t)nx * ny;
    c->prec = precision;
    c->elem = precision / 8;
    const size_t need = fvnl_workspace_bytes(nx, ny, precision);
    if (workspace) {
        if (workspace_bytes < need || ((size_t)workspace & 255)) { delete c; return FVNL_EALLOC; }
        c->ws = workspace;
    } else {
        if (cudaMalloc(&c->ws, need) != cudaSuccess) { (void)cudaGetLastError(); delete c; return FVNL_EALLOC; }
        c->own_ws = true;
    }
    const size_t plane = align_up(c->n * c->elem, 256);
    char* p = (char*)c->ws;
    c->clk = (Clock*)p;
    p += CLOCK_BYTES;
    for (int b = 0; b < 2; ++b)
        for (int k = 0; k < 3; ++k) { c->buf[b][k] = p; p += plane; }
    c->src = (double*)p;
    if (cudaMallocHost((void**)&c->host_clk, sizeof(Clock)) != cudaSuccess) {
        (void)cudaGetLastError();
        if (c->own_ws) cudaFree(c->ws);
        delete c;
        return FVNL_EALLOC;
    }
    std::memset(&c->snap, 0, sizeof(Clock));
    bool ok = cudaMemsetAsync(c->clk, 0, CLOCK_BYTES, c->stream) == cudaSuccess;
    // equilibrium state: q = (1, 0, 0), stored in fp32 contexts as (rho', q2, q3) = (0, 0, 0)
    ok = ok && cudaMemsetAsync(c->buf[0][0], 0, plane, c->stream) == cudaSuccess;
    ok = ok && cudaMemsetAsync(c->buf[0][1], 0, plane, c->stream) == cudaSuccess;
    ok = ok && cudaMemsetAsync(c->buf[0][2], 0, plane, c->stream) == cudaSuccess;
    if (c->prec == 64) k_fill<<<592, 256, 0, c->stream>>>((double*)c->buf[0][0], c->n, 1.0);
    ok = ok && cudaGetLastError() == cudaSuccess;
    c->launches = 1;
    c->have_state = true;
    c->need_prepass = true;
    c->kernel = FVNL_KERNEL_DEFAULT;
    c->variant = DEFAULT_VARIANT;
    c->small = 1;
    // per device (function attributes belong to the context of the current device)
    ok = ok && cudaFuncSetAttribute(k_step_ws<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, ws_smem_bytes<double>()) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(k_step_ws<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, ws_smem_bytes<float>()) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(k_step_fused<FUSED_BX, FUSED_MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    fused_smem_bytes<FUSED_BX>()) == cudaSuccess;
    if (!ok) { (void)cudaGetLastError(); fvnl_destroy(c); return FVNL_ECUDA; }
    *out = c;
    return FVNL_OK;
}

extern "C" void fvnl_destroy(fvnl_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    resolve_spans(c);
    delete c->spans;
    for (int k = 0; k < 3; ++k)
        if (c->star[k]) cudaFree(c->star[k]);
    if (c->gexec) cudaGraphExecDestroy(c->gexec);
    if (c->gstream) cudaStreamDestroy(c->gstream);
    if (c->host_clk) cudaFreeHost(c->host_clk);
    if (c->own_ws && c->ws) cudaFree(c->ws);
    (void)cudaGetLastError();
    delete c;
}

extern "C" int fvnl_set_bc(fvnl_ctx* c, int side, int kind, const fvnl_source* s) {
    if (!c || side < 0 || side > 3 || kind < 0 || kind > 3) return FVNL_EARG;
    Side d;
    std::memset(&d, 0, sizeof(d));
    d.kind = kind;
    if (kind == BC_SOURCE) {
        if (!s || s->shape < 0 || s->shape > 2) return FVNL_EARG;
        if (s->shape != SRC_TANH && !(s->freq_hz > 0)) return FVNL_EARG;
        d.shape = s->shape; d.amp = s->amp; d.freq_hz = s->freq_hz; d.focus_m = s->focus_m; d.centre_m = s->centre_m;
        d.half_aperture_m = s->half_aperture_m; d.t0_s = s->t0_s; d.steep = s->steep; d.theta = s->theta;
    }
    c->g.side[side] = d;
    c->gvalid = false;
    if (c->small_cluster > 0) c->small_cluster = 0;                 // (its shared-memory need depends on the SOURCE sides)
    return FVNL_OK;
}

extern "C" int fvnl_set_option(fvnl_ctx* c, int option, int value) {
    if (!c) return FVNL_EARG;
    c->gvalid = false;
    if (option == FVNL_OPT_KERNEL) {
        if (value != FVNL_KERNEL_DEFAULT && value != FVNL_KERNEL_UNFUSED) return FVNL_EARG;
        if (value != FVNL_KERNEL_DEFAULT && c->prec != 64) return FVNL_EARG;      // the comparison paths are fp64 only
        c->kernel = value;
        return FVNL_OK;
    }
    if (option == FVNL_OPT_ROWS_PER_BLOCK) {
        if (value < 0) return FVNL_EARG;
        c->rows_per_block = value;
        return FVNL_OK;
    }
    if (option == FVNL_OPT_VARIANT) {
        if (value < 0 || value >= N_FUSED_VARIANTS || (value != 0 && c->prec != 64)) return FVNL_EARG;
        c->variant = value;
        return FVNL_OK;
    }
    if (option == FVNL_OPT_KERNEL_TIMING) {
        c->timing = value != 0;
        return FVNL_OK;
    }
    if (option == FVNL_OPT_SMALL_GRID) {
        if (value != 0 && value != 1) return FVNL_EARG;
        c->small = value;
        return FVNL_OK;
    }
    return FVNL_EARG;
}

extern "C" int fvnl_set_state(fvnl_ctx* c, const void* q1, const void* q2, const void* q3, int where) {
    if (!c || !q1 || !q2 || !q3 || where < 0 || where > 3) return FVNL_EARG;
    const bool on_device = where & FVNL_ON_DEVICE, as_f64 = (where & FVNL_PLANES_F64) && c->prec == 32;
    if (as_f64 && !on_device) return FVNL_EARG;                   // the conversion runs on the device
    const void* src[3] = {q1, q2, q3};
    if (as_f64) {
        k_to_f32<<<1184, 256, 0, c->stream>>>((const double*)q1, (const double*)q2, (const double*)q3, (float*)c->buf[c->cur][0],
                                             (float*)c->buf[c->cur][1], (float*)c->buf[c->cur][2], c->n);
        c->launches += 1;
    } else {
        const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        for (int k = 0; k < 3; ++k) CK(cudaMemcpyAsync(c->buf[c->cur][k], src[k], c->n * c->elem, kind, c->stream));
    }
    // reset sticky flags and the lagged maximum, keep t (and the step counter): on the device, in stream order
    k_clock_reset<<<1, 1, 0, c->stream>>>(c->clk);
    c->launches += 1;
    c->snap.flags = 0;
    c->snap.Mprev = 0.0;
    if (!on_device) CK(cudaStreamSynchronize(c->stream));          // the host buffers may be reused on return
    CK(cudaGetLastError());
    c->have_state = true;
    c->need_prepass = true;
    return FVNL_OK;
}

extern "C" int fvnl_shift(fvnl_ctx* c, int cells) {
    if (!c || cells < 0 || cells >= c->g.nx) return FVNL_EARG;
    const Grid& g = c->g;
    if (g.side[SIDE_XLO].kind == BC_PERIODIC || g.side[SIDE_XHI].kind == BC_PERIODIC || g.side[SIDE_XHI].kind == BC_REFLECT)
        return FVNL_EARG;
    if (!c->have_state) return FVNL_ESTATE;
    if (cells == 0) return FVNL_OK;
    char** a = c->buf[c->cur];
    char** b = c->buf[c->cur ^ 1];
    const dim3 grd((g.nx + 255) / 256, g.ny);
    if (c->prec == 64)
        k_shift<double><<<grd, 256, 0, c->stream>>>(g, c->clk, cells, (const double*)a[0], (const double*)a[1], (const double*)a[2],
                                                    (double*)b[0], (double*)b[1], (double*)b[2]);
    else
        k_shift<float><<<grd, 256, 0, c->stream>>>(g, c->clk, cells, (const float*)a[0], (const float*)a[1], (const float*)a[2],
                                                   (float*)b[0], (float*)b[1], (float*)b[2]);
    CK(cudaGetLastError());
    c->launches += 1;
    c->cur ^= 1;
    c->g.x0 += cells * g.dx;
    c->gvalid = false;                                             // (a captured graph holds the old frame)
    return FVNL_OK;
}

extern "C" int fvnl_set_clock(fvnl_ctx* c, double t_s, double last_M) {
    if (!c || !(t_s == t_s)) return FVNL_EARG;
    const double M = last_M > 0.0 ? last_M : 0.0;
    k_clock_set<<<1, 1, 0, c->stream>>>(c->clk, t_s, M);
    c->launches += 1;
    CK(cudaGetLastError());
    c->snap.t = t_s;
    c->snap.Mprev = M;
    c->need_prepass = !(last_M > 0.0);
    return FVNL_OK;
}

static int ensure_star(fvnl_ctx* c) {
    if (c->star[0]) return FVNL_OK;
    const size_t bytes = (size_t)(c->g.ny + 4) * c->g.nx * sizeof(double);
    for (int k = 0; k < 3; ++k)
        if (cudaMalloc((void**)&c->star[k], bytes) != cudaSuccess) { (void)cudaGetLastError(); return FVNL_EALLOC; }
    return FVNL_OK;
}

// Fused step: strips of BX columns (BX - 6 produce output) x chunks of `rows` rows.  Launch variants
// (FVNL_OPT_VARIANT): block width and the register budget the compiler was given (blocks per SM).

// Rows per chunk.  All blocks do the same work, so the grid runs as "waves" of `slots` resident blocks: pick the
// number of chunks that maximises  (work in full waves) x (useful rows per marched row):
//     efficiency = blocks / (ceil(blocks / slots) * slots)  *  rows / (rows + 7)
// (7 = the pipeline fill of a chunk: 3 halo rows below, 3 above, 1 for the y-sweep running one row behind).
static int fused_rows(const fvnl_ctx* c, int strips, int slots, int fill = 7) {
    const int ny = c->g.ny;
    if (c->rows_per_block > 0) return c->rows_per_block < ny ? c->rows_per_block : ny;
    int best_rows = ny;
    double best = -1.0;
    const int max_chunks = ny / 16 > 0 ? ny / 16 : 1;               // chunks not shorter than 16 rows
    for (int chunks = 1; chunks <= max_chunks && chunks <= 4096; ++chunks) {
        const int rows = (ny + chunks - 1) / chunks;
        const int nch = (ny + rows - 1) / rows;
        const long blocks = (long)strips * nch;
        const long waves = (blocks + slots - 1) / slots;
        const double eff = (double)blocks / (double)(waves * slots) * rows / (rows + (double)fill);
        if (eff > best + 1e-9) { best = eff; best_rows = rows; }
    }
    return best_rows;
}

// value / mode / more: what the block that finishes last needs to end the step (step_tail).
static void launch_step(fvnl_ctx* c, char** a, char** b, double value, int mode, int more) {
    const Grid& g = c->g;
    SpanGuard sp(c, FVNL_TIMED_STEP);
    if (c->variant == 0) {
        const int strips = (g.nx + (WS_COLS - 6) - 1) / (WS_COLS - 6);
        const int per_sm = c->prec == 64 ? WsBudget<double>::blocks_per_sm : WsBudget<float>::blocks_per_sm;
        const int rows = fused_rows(c, strips, 148 * per_sm, 9);
        const dim3 grd(strips, (g.ny + rows - 1) / rows);
        // programmatic dependent launch: the grid may be scheduled while the previous step's is still running; it waits for
        // that grid's completion itself (griddepcontrol.wait in the kernel) before it touches global memory
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grd; cfg.blockDim = dim3(256); cfg.stream = c->stream;
        cfg.dynamicSmemBytes = c->prec == 64 ? ws_smem_bytes<double>() : ws_smem_bytes<float>();
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        if (c->prec == 64)
            cudaLaunchKernelEx(&cfg, k_step_ws<double>, g, c->clk, (const double*)a[0], (const double*)a[1], (const double*)a[2],
                               (double*)b[0], (double*)b[1], (double*)b[2], rows, value, mode, more);
        else
            cudaLaunchKernelEx(&cfg, k_step_ws<float>, g, c->clk, (const float*)a[0], (const float*)a[1], (const float*)a[2],
                               (float*)b[0], (float*)b[1], (float*)b[2], rows, value, mode, more);
    } else {
        const int strips = (g.nx + (FUSED_BX - 6) - 1) / (FUSED_BX - 6);
        const int rows = fused_rows(c, strips, 148 * FUSED_MINB);
        const dim3 grd(strips, (g.ny + rows - 1) / rows);
        k_step_fused<FUSED_BX, FUSED_MINB><<<grd, FUSED_BX, fused_smem_bytes<FUSED_BX>(), c->stream>>>(
            g, c->clk, (const double*)a[0], (const double*)a[1], (const double*)a[2], (double*)b[0], (double*)b[1],
            (double*)b[2], rows, value, mode, more);
    }
}

static int read_clock(fvnl_ctx* c) {
    CK(cudaMemcpyAsync(c->host_clk, c->clk, sizeof(Clock), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    c->snap = *c->host_clk;
    return FVNL_OK;
}

static const size_t GRAPH_MAX_CELLS = 1u << 18;      // below this a step is a few microseconds: launches dominate

static void launch_sources(fvnl_ctx* c) {
    const size_t recs = src_off(c->g.nx, c->g.ny, 4) / 3;
    k_sources<<<(unsigned)((recs + 127) / 128), 128, 0, c->stream>>>(c->g, c->clk);
    c->launches += 1;
}

// One time step of the one-pass path on c->stream: ONE launch.  The step kernel's blocks also write the analytic ghost
// cells of the step that follows (into the other buffer), and the block that finishes last ends the step (clock); only
// the first step of a call gets its ghost cells from k_sources (the clock may have been set by the host in between).
static void onepass_step(fvnl_ctx* c, double value, int mode, int more) {
    char** a = c->buf[c->cur];
    char** b = c->buf[c->cur ^ 1];
    launch_step(c, a, b, value, mode, more);
    c->cur ^= 1;
    c->launches += 1;
}

// Small grids: all `nsteps` steps in one launch of one thread-block cluster (fvnl_small.cuh).  Returns false when the
// device does not take such a launch (the caller then runs the per-step path).
static void small_config(cudaLaunchConfig_t* cfg, cudaLaunchAttribute* at, const fvnl_ctx* c, int cs) {
    *cfg = cudaLaunchConfig_t{};
    cfg->gridDim = dim3(cs); cfg->blockDim = dim3(SMALL_THREADS + 32); cfg->stream = c->stream;
    cfg->dynamicSmemBytes = small_smem_bytes(c->g.nx, c->g.ny, cs, c->g.src != nullptr);
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg->attrs = at; cfg->numAttrs = 1;
}

// CTAs of the cluster: the smallest power of two that gives every cell of the largest sub-step a thread of its own, up to
// the largest cluster the device schedules (16 = non-portable size, else 8) with the shared memory the state then needs.
static int small_cluster_size(fvnl_ctx* c) {
    if (c->small_cluster != 0) return c->small_cluster > 0 ? c->small_cluster : 0;
    c->small_cluster = -1;
    (void)cudaFuncSetAttribute(k_steps_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    (void)cudaFuncSetAttribute(k_steps_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, SMALL_MAX_SMEM);
    (void)cudaGetLastError();
    int want = 1;
    while (want < SMALL_MAX_CLUSTER && want * SMALL_THREADS < c->g.nx * (c->g.ny + 4)) want *= 2;
    for (int cs = want; cs >= 1; cs /= 2) {
        if (small_smem_bytes(c->g.nx, c->g.ny, cs, c->g.src != nullptr) > (size_t)SMALL_MAX_SMEM) continue;
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute at[1];
        small_config(&cfg, at, c, cs);
        int ncl = 0;
        if (cudaOccupancyMaxActiveClusters(&ncl, k_steps_cluster, &cfg) == cudaSuccess && ncl >= 1) { c->small_cluster = cs; break; }
        (void)cudaGetLastError();
    }
    return c->small_cluster > 0 ? c->small_cluster : 0;
}

static bool small_steps(fvnl_ctx* c, long nsteps, double value, int mode) {
    const int cs = small_cluster_size(c);
    if (cs < 1) return false;
    int logc = 0;
    while ((1 << logc) < cs) ++logc;
    double** q = (double**)c->buf[c->cur];
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute at[1];
    small_config(&cfg, at, c, cs);
    if (cudaLaunchKernelEx(&cfg, k_steps_cluster, c->g, c->clk, q[0], q[1], q[2], logc, (long long)nsteps, value, mode) !=
        cudaSuccess) {
        (void)cudaGetLastError();
        c->small_cluster = -1;
        return false;
    }
    c->launches += 1;                                               // the state stays in buf[cur]
    return true;
}

extern "C" int fvnl_step(fvnl_ctx* c, long nsteps, double value, int mode) {
    if (!c || nsteps < 0 || !(value > 0.0) || (mode != 0 && mode != 1)) return FVNL_EARG;
    if (!c->have_state) return FVNL_ESTATE;
    bool has_src = false;
    for (int s = 0; s < 4; ++s) has_src = has_src || c->g.side[s].kind == BC_SOURCE;
    c->g.src = has_src ? c->src : nullptr;
    const Grid& g = c->g;
    for (int ax = 0; ax < 2; ++ax)
        if ((g.side[2 * ax].kind == BC_PERIODIC) != (g.side[2 * ax + 1].kind == BC_PERIODIC)) return FVNL_EARG;
    if (mode == 0 && g.delta * value / (g.dx * g.dx) + g.delta * value / (g.dy * g.dy) > 0.5) return FVNL_EARG;
    if (nsteps == 0) return c->snap.flags;
    cudaStream_t st = c->stream;
    if (has_src) launch_sources(c);                                 // analytic ghost cells at t_n of the first step
    const int pre = (mode == 1 && c->need_prepass) ? 1 : 0;
    if (pre) {                                                      // O7: M of the current state (k_clock_reset / _set
        const dim3 grd((g.nx + 1 + 123) / 124, (g.ny + PRE_ROWS - 1) / PRE_ROWS);      // left the running maxima at zero)
        char** q = c->buf[c->cur];
        if (c->prec == 64) k_prepass<double><<<grd, 128, 0, st>>>(g, c->clk, (const double*)q[0], (const double*)q[1], (const double*)q[2]);
        else k_prepass<float><<<grd, 128, 0, st>>>(g, c->clk, (const float*)q[0], (const float*)q[1], (const float*)q[2]);
        c->launches += 1;
    }
    k_clock_begin<<<1, 1, 0, st>>>(g, c->clk, value, mode, pre);
    c->launches += 1;
    c->need_prepass = false;                                        // from here on M_{n-1} is the last step's (reading A7)
    if (c->kernel == FVNL_KERNEL_UNFUSED) {
        const int rc = ensure_star(c);
        if (rc) return rc;
    }
    long n = 0;
    // Small grids: one cluster launch for the whole call.
    if (c->small && c->kernel == FVNL_KERNEL_DEFAULT && c->variant == DEFAULT_VARIANT && c->prec == 64 && !c->timing &&
        c->n <= SMALL_MAX_CELLS && small_steps(c, nsteps, value, mode))
        n = nsteps;
    // Launch-bound grids: replay a captured graph of two steps (A -> B -> A) while at least three steps remain; the last
    // steps (the final one computes no dt for a successor) go out as plain launches below.
    if (n == 0 && c->kernel == FVNL_KERNEL_DEFAULT && !c->timing && c->n <= GRAPH_MAX_CELLS && nsteps >= 4) {
        if (!c->gvalid || c->gvalue != value || c->gmode != mode || c->gcur != c->cur || c->gvariant != c->variant ||
            c->grows != c->rows_per_block) {
            if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
            c->gvalid = false;
            if (!c->gstream && cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking) != cudaSuccess) c->gstream = nullptr;
            cudaGraph_t graph = nullptr;
            if (c->gstream && cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeRelaxed) == cudaSuccess) {
                const cudaStream_t user = c->stream;
                c->stream = c->gstream;
                const long l0 = c->launches;
                for (int half = 0; half < 2; ++half) onepass_step(c, value, mode, 1);
                c->launches = l0;                               // nothing ran: the capture only records
                c->stream = user;
                if (cudaStreamEndCapture(c->gstream, &graph) == cudaSuccess && graph &&
                    cudaGraphInstantiate(&c->gexec, graph, 0) == cudaSuccess) {
                    c->gvalid = true; c->gvalue = value; c->gmode = mode; c->gcur = c->cur; c->gvariant = c->variant;
                    c->grows = c->rows_per_block;
                }
                if (graph) cudaGraphDestroy(graph);
            }
            (void)cudaGetLastError();
        }
        if (c->gvalid) {
            for (; n + 3 <= nsteps; n += 2) {
                CK(cudaGraphLaunch(c->gexec, st));
                c->launches += 2;
            }
        }
    }
    for (; n < nsteps; ++n) {
        const int more = n + 1 < nsteps ? 1 : 0;
        if (c->kernel == FVNL_KERNEL_DEFAULT) {
            onepass_step(c, value, mode, more);
            continue;
        }
        double* a[3] = {(double*)c->buf[c->cur][0], (double*)c->buf[c->cur][1], (double*)c->buf[c->cur][2]};
        double* b[3] = {(double*)c->buf[c->cur ^ 1][0], (double*)c->buf[c->cur ^ 1][1], (double*)c->buf[c->cur ^ 1][2]};
        const dim3 blk(256), grd((g.nx + 255) / 256, g.ny), grdx((g.nx + 255) / 256, g.ny + 4);
        { SpanGuard sp(c, FVNL_TIMED_XSWEEP);
          k_xsweep_unfused<<<grdx, blk, 0, st>>>(g, c->clk, a[0], a[1], a[2], c->star[0], c->star[1], c->star[2]); }
        { SpanGuard sp(c, FVNL_TIMED_YSWEEP);
          k_ysweep_unfused<<<grd, blk, 0, st>>>(g, c->clk, c->star[0], c->star[1], c->star[2], b[0], b[1], b[2]); }
        { SpanGuard sp(c, FVNL_TIMED_SOURCE);
          k_source_unfused<<<grd, blk, 0, st>>>(g, c->clk, b[0], b[1], b[2], a[0], a[1], a[2]); }
        // result is back in `a`: cur unchanged
        k_clock_end<<<1, 1, 0, st>>>(g, c->clk, value, mode, more);
        c->launches += 4;
    }
    CK(cudaGetLastError());
    const int rc = read_clock(c);
    if (rc) return rc;
    // M of the last step is known: a following CFL-mode call continues without a pre-pass (restartable, P10)
    return c->snap.flags;
}

extern "C" int fvnl_get_state(fvnl_ctx* c, void* q1, void* q2, void* q3, int where) {
    if (!c || !q1 || !q2 || !q3 || where < 0 || where > 3) return FVNL_EARG;
    if (!c->have_state) return FVNL_ESTATE;
    const bool on_device = where & FVNL_ON_DEVICE, as_f64 = (where & FVNL_PLANES_F64) && c->prec == 32;
    if (as_f64 && !on_device) return FVNL_EARG;
    void* dst[3] = {q1, q2, q3};
    if (as_f64) {
        k_from_f32<<<1184, 256, 0, c->stream>>>((const float*)c->buf[c->cur][0], (const float*)c->buf[c->cur][1],
                                               (const float*)c->buf[c->cur][2], (double*)q1, (double*)q2, (double*)q3, c->n);
        c->launches += 1;
        CK(cudaGetLastError());
        return FVNL_OK;
    }
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    for (int k = 0; k < 3; ++k) CK(cudaMemcpyAsync(dst[k], c->buf[c->cur][k], c->n * c->elem, kind, c->stream));
    if (!on_device) CK(cudaStreamSynchronize(c->stream));
    return FVNL_OK;
}

extern "C" int fvnl_get_info(fvnl_ctx* c, double* t_s, double* last_dt_s, double* last_cfl, double* last_M, long* steps) {
    if (!c) return FVNL_EARG;
    const int rc = read_clock(c);
    if (rc) return rc;
    if (t_s) *t_s = c->snap.t;
    if (last_dt_s) *last_dt_s = c->snap.last_dt;
    if (last_cfl) *last_cfl = c->snap.last_cfl;
    if (last_M) *last_M = c->snap.Mprev;
    if (steps) *steps = (long)c->snap.steps;
    return FVNL_OK;
}

extern "C" int fvnl_get_kernel_time(fvnl_ctx* c, int which, double* total_ms, long* launches) {
    if (!c || which < 0 || which >= FVNL_TIMED_KINDS) return FVNL_EARG;
    CK(cudaStreamSynchronize(c->stream));
    resolve_spans(c);
    if (total_ms) *total_ms = c->span_ms[which];
    if (launches) *launches = c->span_n[which];
    c->span_ms[which] = 0.0;
    c->span_n[which] = 0;
    return FVNL_OK;
}

// FP64-pipe probe: 8 independent DFMA chains per thread, 16 warps per SM, no memory traffic.
__global__ void __launch_bounds__(128) k_probe_dfma(double* out, int iters, double a, double b) {
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = a + i + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = fma(x[i], b, a);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 12345.678) out[0] = s;                       // never true: keeps the chains alive
}

extern "C" int fvnl_probe_fp64(void* cuda_stream, double* tflops) {
    if (!tflops) return FVNL_EARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* d = nullptr;
    CK(cudaMalloc((void**)&d, 8));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    const int iters = 8192, blocks = sms * 4, threads = 128;
    k_probe_dfma<<<blocks, threads, 0, st>>>(d, 64, 1.0000001, 0.9999999);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, st);
        k_probe_dfma<<<blocks, threads, 0, st>>>(d, iters, 1.0000001, 0.9999999);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { (void)cudaGetLastError(); cudaFree(d); return FVNL_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    *tflops = 2.0 * (double)blocks * threads * iters * 64.0 / (best * 1e-3) / 1e12;
    return FVNL_OK;
}

extern "C" long fvnl_kernel_launches(const fvnl_ctx* c) { return c ? c->launches : 0; }

// ---------------------------------------------------------------------------------------------------------------
// fvnl_step_noalloc: one fixed-dt step by the three-pass kernels with its scratch (clock block, Q* on the y-extended mesh,
// Q**) in a file-scope device array -- no context, no workspace, no allocation (include/fvnl.h).  Every GPU that loads the
// library holds the array until the process exits.  In host code `noalloc_scratch` is a host-side stand-in for the array,
// NOT a device address: its device address is resolved once per device with cudaGetSymbolAddress and that pointer is what
// the kernels get.
static __device__ __align__(256) unsigned char noalloc_scratch[FVNL_NOALLOC_MAX_BYTES];
static const int NOALLOC_CLOCK_DOUBLES = 64;                  // the clock block (sizeof(Clock) <= 512 bytes), 256-aligned
static_assert(sizeof(Clock) <= NOALLOC_CLOCK_DOUBLES * sizeof(double), "clock block");
static const int NOALLOC_MAX_DEVICES = 64;
static unsigned char* noalloc_ptr[NOALLOC_MAX_DEVICES];      // device address of noalloc_scratch, per device (0: not resolved)

// The clock of one stand-alone step: everything that must start at zero is cleared here (the array keeps the previous
// call's contents), then t and the fixed dt with what derives from it.
__global__ void k_noalloc_begin(Grid g, Clock* c, double t, double dt) {
    c->flags = 0;
    c->Mprev = 0.0;
    c->last_dt = c->last_cfl = 0.0;
    c->steps = 0;
    c->t = t;
    clock_set_dt(g, c, dt, 0, 0.0);                            // (also clears the running maxima and the ticket)
}
// End of the step: nu of the step (FVNL_ECFL if > 1) and the flag word for the caller.
__global__ void k_noalloc_end(Grid g, Clock* c, double dt, int* flags_out) {
    clock_advance(g, c, dt, 0, 0);
    if (flags_out) *flags_out = c->flags;
}

extern "C" int fvnl_step_noalloc(int nx, int ny, double dx, double dy, const fvnl_medium* m, const int bc_kind[4],
                                 const fvnl_source* const bc_source[4], double t, double dt, const double* q1_in,
                                 const double* q2_in, const double* q3_in, double* q1_out, double* q2_out, double* q3_out,
                                 int* flags_dev, void* cuda_stream) {
    if (nx < 4 || ny < 4 || !(dx > 0) || !(dy > 0) || !m || !(m->c0 > 0) || !(m->rho0 > 0) || !(m->beta >= 1) ||
        !(m->delta >= 0) || !bc_kind || !(dt > 0.0) || !(t == t))
        return FVNL_EARG;
    if (!q1_in || !q2_in || !q3_in || !q1_out || !q2_out || !q3_out || q1_in == q1_out || q2_in == q2_out || q3_in == q3_out)
        return FVNL_EARG;
    Grid g;
    std::memset(&g, 0, sizeof(g));
    g.nx = nx; g.ny = ny; g.dx = dx; g.dy = dy; g.c0 = m->c0; g.beta = m->beta; g.delta = m->delta;
    for (int sd = 0; sd < 4; ++sd) {
        const int kind = bc_kind[sd];
        if (kind < 0 || kind > 3) return FVNL_EARG;
        g.side[sd].kind = kind;
        if (kind == BC_SOURCE) {
            const fvnl_source* s = bc_source ? bc_source[sd] : nullptr;
            if (!s || s->shape < 0 || s->shape > 2) return FVNL_EARG;
            if (s->shape != SRC_TANH && !(s->freq_hz > 0)) return FVNL_EARG;
            Side& d = g.side[sd];
            d.shape = s->shape; d.amp = s->amp; d.freq_hz = s->freq_hz; d.focus_m = s->focus_m; d.centre_m = s->centre_m;
            d.half_aperture_m = s->half_aperture_m; d.t0_s = s->t0_s; d.steep = s->steep; d.theta = s->theta;
        }
    }
    for (int ax = 0; ax < 2; ++ax)
        if ((g.side[2 * ax].kind == BC_PERIODIC) != (g.side[2 * ax + 1].kind == BC_PERIODIC)) return FVNL_EARG;
    if (g.delta * dt / (dx * dx) + g.delta * dt / (dy * dy) > 0.5) return FVNL_EARG;
    // ---- the scratch: [clock | Q* 3 x (ny+4) x nx | Q** 3 x ny x nx], doubles
    const size_t n = (size_t)nx * ny, nstar = (size_t)nx * (ny + 4);
    const size_t need = (NOALLOC_CLOCK_DOUBLES + 3 * nstar + 3 * n) * sizeof(double);
    if (need > (size_t)FVNL_NOALLOC_MAX_BYTES) return FVNL_ESIZE;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NOALLOC_MAX_DEVICES) { (void)cudaGetLastError(); return FVNL_ECUDA; }
    if (!noalloc_ptr[dev]) {                                       // once per device, with that device current
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, noalloc_scratch) != cudaSuccess || !p) { (void)cudaGetLastError(); return FVNL_ECUDA; }
        noalloc_ptr[dev] = (unsigned char*)p;
    }
    double* base = reinterpret_cast<double*>(noalloc_ptr[dev]);
    Clock* clk = reinterpret_cast<Clock*>(base);
    double* s1 = base + NOALLOC_CLOCK_DOUBLES, *s2 = s1 + nstar, *s3 = s2 + nstar;      // Q*
    double* b1 = s3 + nstar, *b2 = b1 + n, *b3 = b2 + n;                                // Q**
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const dim3 blk(256), grd((nx + 255) / 256, ny), grdx((nx + 255) / 256, ny + 4);
    k_noalloc_begin<<<1, 1, 0, st>>>(g, clk, t, dt);
    k_xsweep_unfused<<<grdx, blk, 0, st>>>(g, clk, q1_in, q2_in, q3_in, s1, s2, s3);
    k_ysweep_unfused<<<grd, blk, 0, st>>>(g, clk, s1, s2, s3, b1, b2, b3);
    k_source_unfused<<<grd, blk, 0, st>>>(g, clk, b1, b2, b3, q1_out, q2_out, q3_out);
    k_noalloc_end<<<1, 1, 0, st>>>(g, clk, dt, flags_dev);
    if (cudaGetLastError() != cudaSuccess) return FVNL_ECUDA;
    return FVNL_OK;
}

extern "C" const char* fvnl_strerror(int code) {
    switch (code) {
        case FVNL_OK: return "ok";
        case FVNL_EARG: return "bad argument";
        case FVNL_EALLOC: return "workspace too small or allocation failed";
        case FVNL_ECUDA: return "CUDA error or no device";
        case FVNL_ESTATE: return "call order: no state set";
        case FVNL_ESIZE: return "grid too large for the static scratch array of fvnl_step_noalloc (FVNL_NOALLOC_MAX_BYTES)";
        default: break;
    }
    if (code & ~(FVNL_ECFL | FVNL_ENONREAL | FVNL_ENONPOS | FVNL_ENAN)) return "unknown code";
    static thread_local char buf[96];
    std::snprintf(buf, sizeof(buf), "device flags:%s%s%s%s", (code & FVNL_ECFL) ? " CFL>1" : "",
                  (code & FVNL_ENONREAL) ? " non-real-eigenvalue" : "", (code & FVNL_ENONPOS) ? " q1<=0" : "",
                  (code & FVNL_ENAN) ? " NaN" : "");
    return buf;
}
