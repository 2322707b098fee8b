// kh_api.cu -- the C-ABI of include/kratos_hydro.h: argument checking, memory, launches.
// No arithmetic of the method lives here; every step of the path runs in the kernels of
// kh_tma.cuh (3D mixed precision: the bench kernel), kh_strip.cuh (2D mixed precision), kh_pair.cuh (mixed
// precision, other blocks with active x and y), kh_tiled.cuh (all-fp64), kh_simple.cuh (any axes), kh_vanleer.cuh (van Leer integrator, general
// blocks) and kh_reduce.cuh (CFL rate, reference pressure, dt bookkeeping, totals); kh_device.cuh holds the
// shared device functions.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/kratos_hydro.h"
#include "kh_device.cuh"
#include "kh_reduce.cuh"
#include "kh_simple.cuh"
#include "kh_tiled.cuh"
#include "kh_pair.cuh"
#include "kh_tma.cuh"
#include "kh_strip.cuh"
#include "kh_vanleer.cuh"

using namespace kh;

static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                            \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(e_ == cudaErrorMemoryAllocation ? KRATOS_ERR_ALLOC : KRATOS_ERR_CUDA,     \
                        "%s: %s", #expr, cudaGetErrorString(e_));                                 \
    } while (0)

enum { SLOT_STAGE1 = 0, SLOT_STAGE2 = 1, SLOT_OTHER = 2 };
enum { CFL_MAX_BLOCKS = 1184 };   // a buffer capacity, not an SM count: p_partial holds 2 * CFL_MAX_BLOCKS doubles: block sums, then block minima

struct kratos_hydro {
    Grid g;
    int prec;        // KRATOS_PREC_*
    int integ;       // 0: Heun, 1: van Leer predictor-corrector
    int variant;     // resolved KRATOS_KERNEL_SIMPLE / _TILED
    bool tiled_ok;   // tiled kernel supports this block
    int zchunk;      // 0 = auto
    tma::StageMaps* maps;  // tensor maps of the TMA kernel (host; NULL when the block is not supported)
    strip::StageMaps* smaps;  // tensor maps of the 2D strip kernel (host; NULL when the block is not supported)
    double* U0;      // current state (device)
    double* U1;      // Heun: predictor state, 5 N fp64.  van Leer: W^{n+1/2}, 5 N float_t primitives (device)
    Ctrl* ctrl;      // device
    Ctrl* h_ctrl;    // pinned host mirror
    dd* partial;     // totals scratch (device)
    double* d_tot;   // 5 doubles (device)
    double* p_partial;  // per-block pressure sums of the cfl kernel (device)
    double* stage_buf;  // Single mode: staging area for the double <-> float conversion of host states (device, on demand)
    int tot_blocks;
    cudaStream_t stream;
    // communication boundaries in z (KRATOS_BC_COMM): ghost arrays [5][2][ny][nx] of the two state arrays beyond the
    // low / high face ([array][side]), the neighbours' ghost arrays this block's stage kernels store into, and what was
    // opened from CUDA IPC handles (closed at destroy)
    bool comm[2];
    double* ghost[2][2];
    double* peer[2][2];
    void* ipc_opened[2][2];
    int device;       // CUDA device the handle lives on (every entry point runs with it current)
    bool rate_valid;  // ctrl->rate_bits holds the rate maximum of U0
    bool pref_valid;  // ctrl->p_ref was computed from the state last given to set_state
    long long launches;
    // profiling: event pairs around the launches of every prof_every-th step (prof_on: this step is one of them)
    bool profiling;
    int prof_every;
    long long prof_step;
    bool prof_on;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<std::pair<int, int>> ev_used;  // (slot, index of start event; stop = +1)
    size_t ev_next;
    double prof_ms[3];
    long long prof_n[3];
};

const char* kratos_hydro_last_error(void) { return g_err; }
const char* kratos_hydro_version(void) { return "kratos-hydro-b200 0.1 (sm_100a)"; }

// ---------------------------------------------------------------------------------------
namespace {

// Makes the handle's device current for the duration of an entry point (a caller may have switched devices
// since create) and restores the caller's device afterwards.
struct DeviceGuard {
    int prev;
    bool switched;
    explicit DeviceGuard(const kratos_hydro* h) : prev(-1), switched(false)
    {
        if (h && cudaGetDevice(&prev) == cudaSuccess && prev != h->device) switched = cudaSetDevice(h->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

struct LaunchTimer {
    kratos_hydro* h;
    int slot;
    int idx;
    LaunchTimer(kratos_hydro* h_, int slot_) : h(h_), slot(slot_), idx(-1)
    {
        h->launches++;
        if (!h->profiling || !h->prof_on) return;
        if (h->ev_next + 2 > h->ev_pool.size()) {
            if (h->ev_pool.size() >= 200000) return;  // stop recording, keep running
            for (int i = 0; i < 2; i++) {
                cudaEvent_t e;
                if (cudaEventCreate(&e) != cudaSuccess) return;
                h->ev_pool.push_back(e);
            }
        }
        idx = (int)h->ev_next;
        h->ev_next += 2;
        cudaEventRecord(h->ev_pool[idx], h->stream);
    }
    ~LaunchTimer()
    {
        if (idx < 0) return;
        cudaEventRecord(h->ev_pool[idx + 1], h->stream);
        h->ev_used.push_back({slot, idx});
    }
};

// called once per step before its launches
void next_step_profiling(kratos_hydro* h)
{
    h->prof_on = !h->profiling || (h->prof_step++ % h->prof_every) == 0;
}

void collect_timing(kratos_hydro* h)
{
    for (auto& u : h->ev_used) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, h->ev_pool[u.second], h->ev_pool[u.second + 1]) == cudaSuccess) {
            h->prof_ms[u.first] += ms;
            h->prof_n[u.first] += 1;
        }
    }
    h->ev_used.clear();
    h->ev_next = 0;
}

int auto_variant(const kratos_hydro* h)
{
    if (h->comm[0] || h->comm[1]) return KRATOS_KERNEL_TMA;   // checked at create: the only kernel that serves them
    if (h->integ == 1) return (h->maps && h->maps->ok) ? KRATOS_KERNEL_TMA : KRATOS_KERNEL_SIMPLE;  // van Leer
    if (h->prec == KRATOS_PREC_SINGLE)   // all-fp32 state: the TMA kernel on float boxes, else the general kernel
        return (h->maps && h->maps->ok) ? KRATOS_KERNEL_TMA : ((h->smaps && h->smaps->ok) ? KRATOS_KERNEL_STRIP : KRATOS_KERNEL_SIMPLE);
    if (!h->tiled_ok) return KRATOS_KERNEL_SIMPLE;
    if (h->prec != KRATOS_PREC_MIXED) return KRATOS_KERNEL_TILED;
    if (h->maps && h->maps->ok) return KRATOS_KERNEL_TMA;
    if (h->smaps && h->smaps->ok) return KRATOS_KERNEL_STRIP;
    return KRATOS_KERNEL_PAIRED;
}

int pick_zchunk(const kratos_hydro* h)
{
    if (h->zchunk > 0 && h->variant == KRATOS_KERNEL_STRIP) return h->zchunk < h->g.n[1] ? h->zchunk : h->g.n[1];
    if (h->zchunk > 0) return h->zchunk < h->g.n[2] ? h->zchunk : h->g.n[2];
    if (h->variant == KRATOS_KERNEL_TMA) return tma::auto_zchunk(h->g);
    if (h->variant == KRATOS_KERNEL_STRIP) return strip::auto_rows(h->g);
    return (h->variant == KRATOS_KERNEL_PAIRED) ? pr::auto_zchunk(h->g) : tiled_auto_zchunk(h->g);
}

template <typename T>
int launch_stage(kratos_hydro* h, int stage)
{
    const Grid& g = h->g;
    const double* Uin = (stage == 1) ? h->U0 : h->U1;
    double* Uout = (stage == 1) ? h->U1 : h->U0;
    LaunchTimer lt(h, stage == 1 ? SLOT_STAGE1 : SLOT_STAGE2);
    if (h->variant == KRATOS_KERNEL_TMA) {
        tma::launch_stage(stage, *h->maps, g, h->ctrl, pick_zchunk(h), h->stream);
    } else if (h->variant == KRATOS_KERNEL_STRIP) {
        strip::launch_stage<double>(stage, *h->smaps, h->U0, Uout, g, h->ctrl, pick_zchunk(h), h->stream);
    } else if (h->variant == KRATOS_KERNEL_PAIRED) {
        pr::launch_stage(stage, Uin, h->U0, Uout, g, h->ctrl, pick_zchunk(h), h->stream);
    } else if (h->variant == KRATOS_KERNEL_TILED) {
        launch_stage_tiled<T>(stage, Uin, h->U0, Uout, g, h->ctrl, pick_zchunk(h), h->stream);
    } else {
        const int threads = 128;
        const long long blocks = (g.N + threads - 1) / threads;
        if (stage == 1)
            stage_simple<T, 1><<<(unsigned)blocks, threads, 0, h->stream>>>(Uin, h->U0, Uout, g, h->ctrl);
        else
            stage_simple<T, 2><<<(unsigned)blocks, threads, 0, h->stream>>>(Uin, h->U0, Uout, g, h->ctrl);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "stage %d launch: %s", stage, cudaGetErrorString(e));
    return KRATOS_OK;
}

// All-fp32 "Single" mode: float2_t = float_t = float; both state arrays hold floats.
int launch_stage_single(kratos_hydro* h, int stage)
{
    const Grid& g = h->g;
    const float* A = reinterpret_cast<const float*>(h->U0);
    float* B = reinterpret_cast<float*>(h->U1);
    LaunchTimer lt(h, stage == 1 ? SLOT_STAGE1 : SLOT_STAGE2);
    const int threads = 128;
    const long long blocks = (g.N + threads - 1) / threads;
    if (h->variant == KRATOS_KERNEL_TMA) tma::launch_stage_single(stage, *h->maps, g, h->ctrl, pick_zchunk(h), h->stream);
    else if (h->variant == KRATOS_KERNEL_STRIP)
        strip::launch_stage<float>(stage, *h->smaps, A, stage == 1 ? B : const_cast<float*>(A), g, h->ctrl, pick_zchunk(h), h->stream);
    else if (stage == 1) stage_simple<float, 1, float><<<(unsigned)blocks, threads, 0, h->stream>>>(A, A, B, g, h->ctrl);
    else            stage_simple<float, 2, float><<<(unsigned)blocks, threads, 0, h->stream>>>(B, A, const_cast<float*>(A), g, h->ctrl);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "stage %d launch: %s", stage, cudaGetErrorString(e));
    return KRATOS_OK;
}

int launch_both_stages(kratos_hydro* h)
{
    int rc;
    if (h->integ == 1) {  // van Leer: predictor into the float_t primitive array, corrector in place
        for (int which = 1; which <= 2; which++) {
            LaunchTimer lt(h, which == 1 ? SLOT_STAGE1 : SLOT_STAGE2);
            const int zc = h->zchunk > 0 ? (h->zchunk < h->g.n[2] ? h->zchunk : h->g.n[2]) : tma::auto_zchunk(h->g);
            const bool on_tma = h->maps && h->maps->ok && h->variant == KRATOS_KERNEL_TMA;   // both sub-steps on the TMA machinery
            if (on_tma && which == 1) tma::launch_vl_predict(*h->maps, h->g, h->ctrl, zc, h->stream);
            else if (on_tma && which == 2) tma::launch_vl_correct(*h->maps, h->g, h->ctrl, zc, h->stream);
            else if (h->prec == KRATOS_PREC_MIXED) vl::launch_step<float>(h->U0, h->U1, h->g, h->ctrl, h->stream, which);
            else                              vl::launch_step<double>(h->U0, h->U1, h->g, h->ctrl, h->stream, which);
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "van Leer sub-step %d launch: %s", which, cudaGetErrorString(e));
        }
        return KRATOS_OK;
    }
    if (h->prec == KRATOS_PREC_SINGLE) {
        if ((rc = launch_stage_single(h, 1))) return rc;
        return launch_stage_single(h, 2);
    }
    if (h->prec == KRATOS_PREC_MIXED) {
        if ((rc = launch_stage<float>(h, 1))) return rc;
        return launch_stage<float>(h, 2);
    }
    if ((rc = launch_stage<double>(h, 1))) return rc;
    return launch_stage<double>(h, 2);
}

int launch_cfl_rate(kratos_hydro* h)
{
    {
        LaunchTimer lt(h, SLOT_OTHER);
        reset_rate_kernel<<<1, 1, 0, h->stream>>>(h->ctrl);
    }
    {
        LaunchTimer lt(h, SLOT_OTHER);
        long long blocks = (h->g.N + 255) / 256;
        if (blocks > CFL_MAX_BLOCKS) blocks = CFL_MAX_BLOCKS;
        if (h->prec == KRATOS_PREC_SINGLE)
            cfl_rate_kernel<float><<<(unsigned)blocks, 256, 0, h->stream>>>(reinterpret_cast<const float*>(h->U0), h->g, h->ctrl, h->p_partial);
        else
            cfl_rate_kernel<double><<<(unsigned)blocks, 256, 0, h->stream>>>(h->U0, h->g, h->ctrl, h->p_partial);
        // the reference pressure is a function of the state given to set_state and of nothing else: calling
        // cfl_dt() between steps must not change what the following steps compute
        if (!h->pref_valid) {
            finish_cfl_kernel<<<1, 1, 0, h->stream>>>(h->ctrl, h->p_partial, (int)blocks, 1.0 / (double)h->g.N);
            h->launches++;
        }
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "cfl launch: %s", cudaGetErrorString(e));
    h->rate_valid = true;
    h->pref_valid = true;
    return KRATOS_OK;
}

__global__ void set_pref_kernel(Ctrl* ctrl, double p_ref) { ctrl->p_ref = p_ref; }

__global__ void configure_run_kernel(Ctrl* ctrl, double cfl, double t_end, double t)
{
    ctrl->cfl = cfl;
    ctrl->t_end = t_end;
    ctrl->t = t;
    ctrl->steps = 0;
    ctrl->nonfinite = 0;
}

int read_ctrl(kratos_hydro* h)
{
    CUDA_TRY(cudaMemcpyAsync(h->h_ctrl, h->ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return KRATOS_OK;
}

// Single mode: the boundary carries doubles, the handle stores floats.  Device buffers are converted directly; host
// buffers go through a device staging area of at most 64 Mi doubles, chunk by chunk.  Synchronises for host buffers.
int convert_state(kratos_hydro* h, double* U, int on_device, bool in)
{
    const long long n = 5 * h->g.N;
    float* S = reinterpret_cast<float*>(h->U0);
    const long long chunk = on_device ? n : (n < (64LL << 20) ? n : (64LL << 20));
    if (!on_device && !h->stage_buf) CUDA_TRY(cudaMalloc(&h->stage_buf, sizeof(double) * (size_t)chunk));
    for (long long o = 0; o < n; o += chunk) {
        const long long m = (n - o < chunk) ? n - o : chunk;
        double* dev = on_device ? U + o : h->stage_buf;
        const unsigned blocks = (unsigned)((m + 255) / 256 < sm_count() * 16 ? (m + 255) / 256 : sm_count() * 16);
        if (in) {
            if (!on_device) CUDA_TRY(cudaMemcpyAsync(dev, U + o, sizeof(double) * (size_t)m, cudaMemcpyHostToDevice, h->stream));
            LaunchTimer lt(h, SLOT_OTHER);
            convert_state_kernel<double, float><<<blocks, 256, 0, h->stream>>>(dev, S + o, m);
        } else {
            {
                LaunchTimer lt(h, SLOT_OTHER);
                convert_state_kernel<float, double><<<blocks, 256, 0, h->stream>>>(S + o, dev, m);
            }
            if (!on_device) CUDA_TRY(cudaMemcpyAsync(U + o, dev, sizeof(double) * (size_t)m, cudaMemcpyDeviceToHost, h->stream));
        }
        if (!on_device) CUDA_TRY(cudaStreamSynchronize(h->stream));   // the staging area is reused by the next chunk
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "state conversion: %s", cudaGetErrorString(e));
    return KRATOS_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------
kratos_hydro_t* kratos_hydro_create(int nx, int ny, int nz, double gamma, int scheme, const int bc[6])
{
    g_err[0] = 0;
    const int n[3] = {nx, ny, nz};
    if (!bc) { fail(KRATOS_ERR_ARG, "bc is NULL"); return nullptr; }
    if (!(gamma > 1.0) || !std::isfinite(gamma)) { fail(KRATOS_ERR_ARG, "gamma must be > 1"); return nullptr; }
    const int prec = scheme & 3, integ = (scheme >> 4) & 3;
    if (prec > KRATOS_PREC_SINGLE || integ > 1 || (scheme & ~0x33) || (prec == KRATOS_PREC_SINGLE && integ != 0)) {
        fail(KRATOS_ERR_ARG, "unsupported scheme word 0x%x", scheme);
        return nullptr;
    }
    int nactive = 0;
    for (int d = 0; d < 3; d++) {
        if (n[d] < 1 || (n[d] > 1 && n[d] < 4)) {
            fail(KRATOS_ERR_ARG, "extent %d of axis %d: active axes need >= 4 cells", n[d], d);
            return nullptr;
        }
        if (n[d] > 1) {
            nactive++;
            const int lo = bc[2 * d], hi = bc[2 * d + 1];
            const int top = (d == 2) ? KRATOS_BC_COMM : KRATOS_BC_REFLECT;   // communication boundaries: z faces only
            if (lo < 0 || lo > top || hi < 0 || hi > top) { fail(KRATOS_ERR_ARG, "bad bc code on axis %d", d); return nullptr; }
            if ((lo == KRATOS_BC_PERIODIC) != (hi == KRATOS_BC_PERIODIC)) {
                fail(KRATOS_ERR_ARG, "periodic on one side only of axis %d", d);
                return nullptr;
            }
        }
    }
    if (nactive == 0) { fail(KRATOS_ERR_ARG, "no active axis"); return nullptr; }
    if ((long long)nx * ny >= (1LL << 31) || (long long)nx * ny * nz >= (1LL << 40)) {
        fail(KRATOS_ERR_ARG, "block too large: nx*ny must be < 2^31 cells");
        return nullptr;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        fail(KRATOS_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
        return nullptr;
    }
    kratos_hydro* h = new (std::nothrow) kratos_hydro();
    if (!h) { fail(KRATOS_ERR_ALLOC, "host allocation failed"); return nullptr; }
    Grid& g = h->g;
    g.N = 1;
    for (int d = 0; d < 3; d++) {
        g.n[d] = n[d];
        g.active[d] = n[d] > 1;
        g.bc[2 * d] = g.active[d] ? bc[2 * d] : 0;
        g.bc[2 * d + 1] = g.active[d] ? bc[2 * d + 1] : 0;
        g.inv_dx[d] = g.active[d] ? (double)n[d] : 0.0;
        g.N *= n[d];
    }
    g.gamma = gamma;
    h->prec = prec;
    h->integ = integ;
    h->tiled_ok = g.active[0] && g.active[1] && integ == 0;   // the fused stage kernels are the Heun path
    h->maps = nullptr;
    h->smaps = nullptr;
    for (int side = 0; side < 2; side++) {
        h->comm[side] = g.active[2] && g.bc[4 + side] == KRATOS_BC_COMM;
        for (int a = 0; a < 2; a++) { h->ghost[a][side] = nullptr; h->peer[a][side] = nullptr; h->ipc_opened[a][side] = nullptr; }
    }
    if ((h->comm[0] || h->comm[1]) && (prec != KRATOS_PREC_MIXED || integ != 0 || !tma::supported(g) || nz < 4)) {
        fail(KRATOS_ERR_ARG, "communication boundaries need mixed precision, the Heun integrator, three active axes, "
                             "nx %% 32 == 0, ny %% 16 == 0 and nz >= 4 (they are served by the TMA kernel)");
        delete h;
        return nullptr;
    }
    h->variant = auto_variant(h);
    h->zchunk = 0;
    h->stream = 0;
    h->device = 0;
    cudaGetDevice(&h->device);
    h->rate_valid = false;
    h->pref_valid = false;
    h->launches = 0;
    h->profiling = false;
    h->prof_every = 1;
    h->prof_step = 0;
    h->prof_on = true;
    h->ev_next = 0;
    for (int s = 0; s < 3; s++) { h->prof_ms[s] = 0; h->prof_n[s] = 0; }
    h->U0 = h->U1 = nullptr;
    h->ctrl = nullptr; h->h_ctrl = nullptr; h->partial = nullptr; h->d_tot = nullptr; h->p_partial = nullptr;
    h->tot_blocks = (int)((g.N + 255) / 256 < 592 ? (g.N + 255) / 256 : 592);
    const size_t bytes = (prec == KRATOS_PREC_SINGLE ? sizeof(float) : sizeof(double)) * 5 * (size_t)g.N;
    h->stage_buf = nullptr;
    // second array: the fp64 predictor of Heun, or the float_t primitives W^{n+1/2} of van Leer (PAPER.md:272:
    // "saves up to ~1/3 of the device memory": 40 + 20 instead of 40 + 40 bytes per cell in mixed precision)
    const size_t bytes1 = (integ == 1) ? (prec == KRATOS_PREC_MIXED ? sizeof(float) : sizeof(double)) * 5 * (size_t)g.N : bytes;
    cudaError_t e;
    if ((e = cudaMalloc(&h->U0, bytes)) != cudaSuccess || (e = cudaMalloc(&h->U1, bytes1)) != cudaSuccess ||
        (e = cudaMalloc(&h->ctrl, sizeof(Ctrl))) != cudaSuccess ||
        (e = cudaMalloc(&h->partial, sizeof(dd) * 5 * h->tot_blocks)) != cudaSuccess ||
        (e = cudaMalloc(&h->d_tot, sizeof(double) * 5)) != cudaSuccess ||
        (e = cudaMalloc(&h->p_partial, sizeof(double) * 2 * CFL_MAX_BLOCKS)) != cudaSuccess ||
        (e = cudaMallocHost(&h->h_ctrl, sizeof(Ctrl) + 64)) != cudaSuccess ||
        (e = cudaMemset(h->ctrl, 0, sizeof(Ctrl))) != cudaSuccess ||
        (e = cudaMemset(h->U0, 0, bytes)) != cudaSuccess || (e = cudaMemset(h->U1, 0, bytes1)) != cudaSuccess) {
        fail(e == cudaErrorMemoryAllocation ? KRATOS_ERR_ALLOC : KRATOS_ERR_CUDA, "create: %s", cudaGetErrorString(e));
        cudaGetLastError();
        kratos_hydro_destroy(h);
        return nullptr;
    }
    for (int side = 0; side < 2; side++) {
        if (!h->comm[side]) continue;
        const size_t gb = sizeof(double) * 5 * 2 * (size_t)nx * ny;
        for (int a = 0; a < 2; a++) {
            if ((e = cudaMalloc(&h->ghost[a][side], gb)) != cudaSuccess || (e = cudaMemset(h->ghost[a][side], 0, gb)) != cudaSuccess) {
                fail(e == cudaErrorMemoryAllocation ? KRATOS_ERR_ALLOC : KRATOS_ERR_CUDA, "create (ghost planes): %s", cudaGetErrorString(e));
                cudaGetLastError();
                kratos_hydro_destroy(h);
                return nullptr;
            }
        }
    }
    tiled_configure();
    pr::configure();
    tma::configure();
    strip::configure();
    if (prec == KRATOS_PREC_SINGLE && tma::supported(g)) {
        h->maps = new (std::nothrow) tma::StageMaps;
        if (h->maps) tma::build_maps_single(h->maps, reinterpret_cast<const float*>(h->U0), reinterpret_cast<const float*>(h->U1), g);
    }
    if (prec == KRATOS_PREC_MIXED && tma::supported(g)) {
        h->maps = new (std::nothrow) tma::StageMaps;
        if (h->maps && integ == 0) tma::build_maps(h->maps, h->U0, h->U1, g);
        if (h->maps && integ == 1) tma::build_maps_vl(h->maps, h->U0, (const float*)h->U1, g);
    }
    if (prec == KRATOS_PREC_SINGLE && strip::supported_single(g)) {
        h->smaps = new (std::nothrow) strip::StageMaps;
        if (h->smaps) strip::build_maps(h->smaps, reinterpret_cast<const float*>(h->U0), reinterpret_cast<const float*>(h->U1), g);
    }
    if (prec == KRATOS_PREC_MIXED && integ == 0 && strip::supported(g)) {
        h->smaps = new (std::nothrow) strip::StageMaps;
        if (h->smaps) strip::build_maps(h->smaps, (const double*)h->U0, (const double*)h->U1, g);
    }
    if (h->comm[0] || h->comm[1]) {
        double* none[2] = {nullptr, nullptr};
        if (!h->maps || !h->maps->ok || !tma::set_comm_maps(h->maps, g, h->ghost[0], h->ghost[1], none, none)) {
            fail(KRATOS_ERR_CUDA, "create: tensor maps of the ghost planes");
            kratos_hydro_destroy(h);
            return nullptr;
        }
    }
    h->variant = auto_variant(h);
    return h;
}

void kratos_hydro_destroy(kratos_hydro_t* h)
{
    if (!h) return;
    DeviceGuard dg(h);
    cudaFree(h->U0);
    cudaFree(h->U1);
    cudaFree(h->ctrl);
    cudaFree(h->partial);
    cudaFree(h->d_tot);
    cudaFree(h->p_partial);
    cudaFree(h->stage_buf);
    for (int a = 0; a < 2; a++)
        for (int side = 0; side < 2; side++) {
            cudaFree(h->ghost[a][side]);
            if (h->ipc_opened[a][side]) cudaIpcCloseMemHandle(h->ipc_opened[a][side]);
        }
    if (h->h_ctrl) cudaFreeHost(h->h_ctrl);
    delete h->maps;
    delete h->smaps;
    for (auto e : h->ev_pool) cudaEventDestroy(e);
    delete h;
}

int kratos_hydro_set_spacing(kratos_hydro_t* h, double dx, double dy, double dz)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    const double s[3] = {dx, dy, dz};
    for (int d = 0; d < 3; d++)
        if (h->g.active[d] && (!(s[d] > 0.0) || !std::isfinite(s[d]))) return fail(KRATOS_ERR_ARG, "spacing must be > 0");
    for (int d = 0; d < 3; d++) h->g.inv_dx[d] = h->g.active[d] ? 1.0 / s[d] : 0.0;
    h->rate_valid = false;
    return KRATOS_OK;
}

int kratos_hydro_set_stream(kratos_hydro_t* h, void* cuda_stream)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    h->stream = (cudaStream_t)cuda_stream;
    return KRATOS_OK;
}

int kratos_hydro_set_kernel(kratos_hydro_t* h, int variant)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    if (variant == KRATOS_KERNEL_AUTO) variant = auto_variant(h);
    if ((h->comm[0] || h->comm[1]) && variant != KRATOS_KERNEL_TMA)
        return fail(KRATOS_ERR_ARG, "blocks with communication boundaries are served by the TMA kernel only");
    if (h->prec == KRATOS_PREC_SINGLE && variant != auto_variant(h) && variant != KRATOS_KERNEL_SIMPLE)
        return fail(KRATOS_ERR_ARG, "this kernel variant does not serve the all-fp32 mode on this block");
    if ((variant == KRATOS_KERNEL_TILED || variant == KRATOS_KERNEL_PAIRED) && !h->tiled_ok)
        return fail(KRATOS_ERR_ARG, "tiled and paired kernels need active x and y axes");
    if (variant == KRATOS_KERNEL_PAIRED && h->prec != KRATOS_PREC_MIXED)
        return fail(KRATOS_ERR_ARG, "the paired kernel is the mixed-precision path");
    if (variant == KRATOS_KERNEL_TMA && !(h->maps && h->maps->ok))
        return fail(KRATOS_ERR_ARG, "the TMA kernel needs mixed precision, three active axes, nx %% 32 == 0 and ny %% 16 == 0");
    if (variant == KRATOS_KERNEL_STRIP && !(h->smaps && h->smaps->ok))
        return fail(KRATOS_ERR_ARG, "the strip kernel needs mixed precision, the Heun integrator and a 2D block (nz = 1) with even nx, ny");
    if (variant != KRATOS_KERNEL_SIMPLE && variant != KRATOS_KERNEL_TILED && variant != KRATOS_KERNEL_PAIRED &&
        variant != KRATOS_KERNEL_TMA && variant != KRATOS_KERNEL_STRIP)
        return fail(KRATOS_ERR_ARG, "bad variant");
    h->variant = variant;
    return KRATOS_OK;
}

int kratos_hydro_get_kernel(kratos_hydro_t* h, int* variant)
{
    if (!h || !variant) return fail(KRATOS_ERR_ARG, "NULL argument");
    *variant = h->variant;
    return KRATOS_OK;
}

int kratos_hydro_set_zchunk(kratos_hydro_t* h, int planes)
{
    if (!h || planes < 0) return fail(KRATOS_ERR_ARG, "bad argument");
    h->zchunk = planes;
    return KRATOS_OK;
}

int kratos_hydro_set_state(kratos_hydro_t* h, const double* U, int on_device)
{
    if (!h || !U) return fail(KRATOS_ERR_ARG, "NULL argument");
    const size_t bytes = sizeof(double) * 5 * (size_t)h->g.N;
    DeviceGuard dg(h);
    if (h->prec == KRATOS_PREC_SINGLE) {
        int rc = convert_state(h, const_cast<double*>(U), on_device, true);
        if (rc) return rc;
    } else {
        CUDA_TRY(cudaMemcpyAsync(h->U0, U, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
        if (!on_device) CUDA_TRY(cudaStreamSynchronize(h->stream));
    }
    h->rate_valid = false;
    h->pref_valid = false;
    return KRATOS_OK;
}

int kratos_hydro_get_state(kratos_hydro_t* h, double* U, int on_device)
{
    if (!h || !U) return fail(KRATOS_ERR_ARG, "NULL argument");
    const size_t bytes = sizeof(double) * 5 * (size_t)h->g.N;
    DeviceGuard dg(h);
    if (h->prec == KRATOS_PREC_SINGLE) return convert_state(h, U, on_device, false);
    CUDA_TRY(cudaMemcpyAsync(U, h->U0, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    if (!on_device) CUDA_TRY(cudaStreamSynchronize(h->stream));
    return KRATOS_OK;
}

int kratos_hydro_cfl_dt(kratos_hydro_t* h, double cfl, double* dt_out)
{
    if (!h || !dt_out) return fail(KRATOS_ERR_ARG, "NULL argument");
    if (!(cfl > 0.0) || !std::isfinite(cfl)) return fail(KRATOS_ERR_ARG, "cfl must be > 0");
    DeviceGuard dg(h);
    int rc;
    if ((rc = launch_cfl_rate(h))) return rc;
    if ((rc = read_ctrl(h))) return rc;
    double rate;
    memcpy(&rate, &h->h_ctrl->rate_bits, sizeof(double));
    const double dt = cfl / rate;
    *dt_out = dt;
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(KRATOS_ERR_NONFINITE, "non-finite CFL time step (rate %g)", rate);
    return KRATOS_OK;
}

int kratos_hydro_step(kratos_hydro_t* h, double dt)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(KRATOS_ERR_ARG, "dt must be > 0 and finite");
    if (h->comm[0] || h->comm[1])
        return fail(KRATOS_ERR_ARG, "a block with communication boundaries advances by kratos_hydro_substep (its neighbours must "
                                    "have delivered their planes between the stages)");
    DeviceGuard dg(h);
    int rc;
    // first step after set_state: the reference pressure of the mixed-precision kernels comes from this state
    if (!h->pref_valid && h->prec == KRATOS_PREC_MIXED && (rc = launch_cfl_rate(h))) return rc;
    next_step_profiling(h);
    {
        LaunchTimer lt(h, SLOT_OTHER);
        set_dt_kernel<<<1, 1, 0, h->stream>>>(h->ctrl, dt);
    }
    if ((rc = launch_both_stages(h))) return rc;
    h->rate_valid = true;  // stage 2 left the rate maximum of the new state in ctrl
    return KRATOS_OK;
}

static int run_impl(kratos_hydro_t* h, double cfl, double t_end, int max_steps, double* t_inout, int* steps_done)
{
    if (!h || !t_inout) return fail(KRATOS_ERR_ARG, "NULL argument");
    if (!(cfl > 0.0) || !std::isfinite(cfl) || max_steps < 0) return fail(KRATOS_ERR_ARG, "bad cfl / step count");
    if (!std::isfinite(*t_inout) || !std::isfinite(t_end)) return fail(KRATOS_ERR_ARG, "non-finite time");
    if (h->comm[0] || h->comm[1])
        return fail(KRATOS_ERR_ARG, "a block with communication boundaries advances by kratos_hydro_substep");
    DeviceGuard dg(h);
    int rc;
    {
        LaunchTimer lt(h, SLOT_OTHER);
        configure_run_kernel<<<1, 1, 0, h->stream>>>(h->ctrl, cfl, t_end > 0.0 ? t_end : 0.0, *t_inout);
    }
    if ((!h->rate_valid || !h->pref_valid) && (rc = launch_cfl_rate(h))) return rc;
    int done = 0;
    // run_until: steps are enqueued in batches and the host looks at t between batches.  The batch shrinks to
    // the number of steps the last dt predicts are left (+1), so that hardly any zero-length step is enqueued
    // after t has reached t_end.
    int batch = (t_end > 0.0) ? 8 : max_steps;
    while (done < max_steps) {
        const int nb = (max_steps - done < batch) ? max_steps - done : batch;
        for (int s = 0; s < nb; s++) {
            next_step_profiling(h);
            {
                LaunchTimer lt(h, SLOT_OTHER);
                prepare_step_kernel<<<1, 1, 0, h->stream>>>(h->ctrl);
            }
            if ((rc = launch_both_stages(h))) return rc;
        }
        done += nb;
        if ((rc = read_ctrl(h))) return rc;
        if (h->h_ctrl->nonfinite) break;
        if (t_end > 0.0) {
            if (h->h_ctrl->t >= t_end) break;
            const double left = (t_end - h->h_ctrl->t) / (h->h_ctrl->dt > 0.0 ? h->h_ctrl->dt : t_end);
            batch = left > 63.0 ? 64 : (int)left + 1;
        }
    }
    if (done == 0 && (rc = read_ctrl(h))) return rc;
    *t_inout = h->h_ctrl->t;
    if (steps_done) *steps_done = (int)h->h_ctrl->steps;
    h->rate_valid = !h->h_ctrl->nonfinite;
    if (h->h_ctrl->nonfinite) return fail(KRATOS_ERR_NONFINITE, "non-finite time step during run (t = %g)", h->h_ctrl->t);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "run: %s", cudaGetErrorString(e));
    return KRATOS_OK;
}

int kratos_hydro_run(kratos_hydro_t* h, double cfl, int nsteps, double* t_inout)
{
    return run_impl(h, cfl, 0.0, nsteps, t_inout, nullptr);
}

int kratos_hydro_run_until(kratos_hydro_t* h, double cfl, double t_end, int max_steps, double* t_inout, int* steps_done)
{
    if (!(t_end > 0.0)) return fail(KRATOS_ERR_ARG, "t_end must be > 0");
    return run_impl(h, cfl, t_end, max_steps, t_inout, steps_done);
}

int kratos_hydro_totals(kratos_hydro_t* h, double out[5])
{
    if (!h || !out) return fail(KRATOS_ERR_ARG, "NULL argument");
    DeviceGuard dg(h);
    {
        LaunchTimer lt(h, SLOT_OTHER);
        if (h->prec == KRATOS_PREC_SINGLE)
            totals_kernel<float><<<dim3(h->tot_blocks, 5), 256, 0, h->stream>>>(reinterpret_cast<const float*>(h->U0), h->g.N, h->partial);
        else
            totals_kernel<double><<<dim3(h->tot_blocks, 5), 256, 0, h->stream>>>(h->U0, h->g.N, h->partial);
    }
    {
        LaunchTimer lt(h, SLOT_OTHER);
        totals_final_kernel<<<1, 32, 0, h->stream>>>(h->partial, h->tot_blocks, h->d_tot);
    }
    double* scratch = reinterpret_cast<double*>(reinterpret_cast<char*>(h->h_ctrl) + sizeof(Ctrl));
    static_assert(sizeof(Ctrl) % 8 == 0, "Ctrl must keep doubles aligned");
    CUDA_TRY(cudaMemcpyAsync(scratch, h->d_tot, sizeof(double) * 5, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (int m = 0; m < 5; m++) out[m] = scratch[m];
    return KRATOS_OK;
}

int kratos_hydro_floor_hits(kratos_hydro_t* h, long long* n)
{
    if (!h || !n) return fail(KRATOS_ERR_ARG, "NULL argument");
    DeviceGuard dg(h);
    int rc = read_ctrl(h);
    if (rc) return rc;
    *n = (long long)h->h_ctrl->floor_hits;
    return KRATOS_OK;
}

int kratos_hydro_status(kratos_hydro_t* h)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    DeviceGuard dg(h);
    int rc = read_ctrl(h);
    if (rc) return rc;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "status: %s", cudaGetErrorString(e));
    if (h->h_ctrl->nonfinite) return fail(KRATOS_ERR_NONFINITE, "a time step came out non-finite (t = %g)", h->h_ctrl->t);
    if (h->rate_valid) {
        // the final kernel of every step reduces the CFL rate of the new state and maps NaN onto +inf
        double rate;
        memcpy(&rate, &h->h_ctrl->rate_bits, sizeof(double));
        if (!(rate < HUGE_VAL)) return fail(KRATOS_ERR_NONFINITE, "non-finite state (CFL rate %g, t = %g)", rate, h->h_ctrl->t);
    }
    return KRATOS_OK;
}

int kratos_hydro_launch_count(kratos_hydro_t* h, long long* n)
{
    if (!h || !n) return fail(KRATOS_ERR_ARG, "NULL argument");
    *n = h->launches;
    return KRATOS_OK;
}

int kratos_hydro_set_profiling(kratos_hydro_t* h, int enable)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    DeviceGuard dg(h);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    h->ev_used.clear();
    h->ev_next = 0;
    for (int s = 0; s < 3; s++) { h->prof_ms[s] = 0; h->prof_n[s] = 0; }
    h->profiling = enable != 0;
    h->prof_every = enable > 1 ? enable : 1;
    h->prof_step = 0;
    h->prof_on = true;
    return KRATOS_OK;
}

int kratos_hydro_get_timing(kratos_hydro_t* h, double ms[3], long long launches[3])
{
    if (!h || !ms || !launches) return fail(KRATOS_ERR_ARG, "NULL argument");
    DeviceGuard dg(h);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    collect_timing(h);
    for (int s = 0; s < 3; s++) { ms[s] = h->prof_ms[s]; launches[s] = h->prof_n[s]; }
    return KRATOS_OK;
}

// ---------------------------------------------------------------------------------------
// Communication boundaries (Sec. 3.1.2) and the pieces of a step a multi-block driver interleaves
// with its own synchronisation (paper_2501_02317_b200/slab.py).

static int check_ghost_args(kratos_hydro_t* h, int array, int side)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    if (array < 0 || array > 1 || side < 0 || side > 1) return fail(KRATOS_ERR_ARG, "array and side must be 0 or 1");
    if (!h->comm[side]) return fail(KRATOS_ERR_ARG, "z face %d of this block is no communication boundary", side);
    return KRATOS_OK;
}

int kratos_hydro_ghost_array(kratos_hydro_t* h, int array, int side, double** ptr)
{
    int rc = check_ghost_args(h, array, side);
    if (rc) return rc;
    if (!ptr) return fail(KRATOS_ERR_ARG, "NULL argument");
    *ptr = h->ghost[array][side];
    return KRATOS_OK;
}

int kratos_hydro_ghost_ipc_handle(kratos_hydro_t* h, int array, int side, unsigned char handle[64])
{
    int rc = check_ghost_args(h, array, side);
    if (rc) return rc;
    if (!handle) return fail(KRATOS_ERR_ARG, "NULL argument");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handles are 64 bytes");
    DeviceGuard dg(h);
    cudaIpcMemHandle_t m;
    CUDA_TRY(cudaIpcGetMemHandle(&m, h->ghost[array][side]));
    memcpy(handle, &m, 64);
    return KRATOS_OK;
}

int kratos_hydro_set_peer(kratos_hydro_t* h, int side, double* peer_ghost_state, double* peer_ghost_pred)
{
    int rc = check_ghost_args(h, 0, side);
    if (rc) return rc;
    if (!peer_ghost_state || !peer_ghost_pred) return fail(KRATOS_ERR_ARG, "NULL peer array");
    DeviceGuard dg(h);
    h->peer[0][side] = peer_ghost_state;
    h->peer[1][side] = peer_ghost_pred;
    double* none[2] = {nullptr, nullptr};
    if (!tma::set_comm_maps(h->maps, h->g, none, none, h->peer[0], h->peer[1]))
        return fail(KRATOS_ERR_CUDA, "tensor maps of the peer ghost arrays");
    return KRATOS_OK;
}

int kratos_hydro_open_peer(kratos_hydro_t* h, int side, const unsigned char handle_state[64], const unsigned char handle_pred[64])
{
    int rc = check_ghost_args(h, 0, side);
    if (rc) return rc;
    if (!handle_state || !handle_pred) return fail(KRATOS_ERR_ARG, "NULL argument");
    DeviceGuard dg(h);
    void* p[2] = {nullptr, nullptr};
    const unsigned char* hd[2] = {handle_state, handle_pred};
    for (int a = 0; a < 2; a++) {
        cudaIpcMemHandle_t m;
        memcpy(&m, hd[a], 64);
        if (h->ipc_opened[a][side]) { cudaIpcCloseMemHandle(h->ipc_opened[a][side]); h->ipc_opened[a][side] = nullptr; }
        CUDA_TRY(cudaIpcOpenMemHandle(&p[a], m, cudaIpcMemLazyEnablePeerAccess));
        h->ipc_opened[a][side] = p[a];
    }
    return kratos_hydro_set_peer(h, side, (double*)p[0], (double*)p[1]);
}

static int peers_ready(kratos_hydro_t* h)
{
    for (int side = 0; side < 2; side++)
        if (h->comm[side] && (!h->peer[0][side] || !h->peer[1][side]))
            return fail(KRATOS_ERR_ARG, "z face %d is a communication boundary without a peer (kratos_hydro_set_peer / _open_peer)", side);
    return KRATOS_OK;
}

int kratos_hydro_push_halo(kratos_hydro_t* h)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    int rc = peers_ready(h);
    if (rc) return rc;
    DeviceGuard dg(h);
    const Grid& g = h->g;
    const size_t plane = (size_t)g.n[0] * g.n[1];
    for (int side = 0; side < 2; side++) {
        if (!h->comm[side]) continue;
        const size_t first = side == 0 ? 0 : (size_t)(g.n[2] - 2) * plane;   // the two planes next to the face
        for (int f = 0; f < 5; f++)
            CUDA_TRY(cudaMemcpyAsync(h->peer[0][side] + (size_t)f * 2 * plane, h->U0 + (size_t)f * g.N + first,
                                     sizeof(double) * 2 * plane, cudaMemcpyDefault, h->stream));
    }
    return KRATOS_OK;
}

int kratos_hydro_begin_run(kratos_hydro_t* h, double cfl, double t0)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    if (!(cfl > 0.0) || !std::isfinite(cfl) || !std::isfinite(t0)) return fail(KRATOS_ERR_ARG, "bad cfl / time");
    DeviceGuard dg(h);
    int rc;
    {
        LaunchTimer lt(h, SLOT_OTHER);
        configure_run_kernel<<<1, 1, 0, h->stream>>>(h->ctrl, cfl, 0.0, t0);
    }
    if ((!h->rate_valid || !h->pref_valid) && (rc = launch_cfl_rate(h))) return rc;
    return KRATOS_OK;
}

int kratos_hydro_substep(kratos_hydro_t* h, int phase)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    if (h->integ != 0 || h->prec == KRATOS_PREC_SINGLE) return fail(KRATOS_ERR_ARG, "substep serves the Heun integrator on an fp64 state");
    DeviceGuard dg(h);
    int rc;
    if (phase == KRATOS_PHASE_PREPARE) {
        if (!h->rate_valid || !h->pref_valid) return fail(KRATOS_ERR_ARG, "substep before kratos_hydro_begin_run");
        next_step_profiling(h);
        LaunchTimer lt(h, SLOT_OTHER);
        prepare_step_kernel<<<1, 1, 0, h->stream>>>(h->ctrl);
        return KRATOS_OK;
    }
    if (phase != KRATOS_PHASE_STAGE1 && phase != KRATOS_PHASE_STAGE2) return fail(KRATOS_ERR_ARG, "bad phase");
    if ((rc = peers_ready(h))) return rc;
    rc = (h->prec == KRATOS_PREC_MIXED) ? launch_stage<float>(h, phase) : launch_stage<double>(h, phase);
    if (rc == KRATOS_OK && phase == KRATOS_PHASE_STAGE2) h->rate_valid = true;
    return rc;
}

int kratos_hydro_end_run(kratos_hydro_t* h, double* t, int* steps_done)
{
    if (!h || !t) return fail(KRATOS_ERR_ARG, "NULL argument");
    DeviceGuard dg(h);
    int rc = read_ctrl(h);
    if (rc) return rc;
    *t = h->h_ctrl->t;
    if (steps_done) *steps_done = (int)h->h_ctrl->steps;
    if (h->h_ctrl->nonfinite) return fail(KRATOS_ERR_NONFINITE, "non-finite time step during run (t = %g)", h->h_ctrl->t);
    return KRATOS_OK;
}

int kratos_hydro_get_rate(kratos_hydro_t* h, double* rate, int on_device)
{
    if (!h || !rate) return fail(KRATOS_ERR_ARG, "NULL argument");
    if (!h->rate_valid) return fail(KRATOS_ERR_ARG, "no CFL rate at hand (kratos_hydro_begin_run / cfl_dt / a stage 2 first)");
    DeviceGuard dg(h);
    CUDA_TRY(cudaMemcpyAsync(rate, &h->ctrl->rate_bits, sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    if (!on_device) CUDA_TRY(cudaStreamSynchronize(h->stream));
    return KRATOS_OK;
}

int kratos_hydro_set_rate(kratos_hydro_t* h, const double* rate, int on_device)
{
    if (!h || !rate) return fail(KRATOS_ERR_ARG, "NULL argument");
    DeviceGuard dg(h);
    CUDA_TRY(cudaMemcpyAsync(&h->ctrl->rate_bits, rate, sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
    if (!on_device) CUDA_TRY(cudaStreamSynchronize(h->stream));
    h->rate_valid = true;
    return KRATOS_OK;
}

int kratos_hydro_get_reference_pressure(kratos_hydro_t* h, double* p_ref)
{
    if (!h || !p_ref) return fail(KRATOS_ERR_ARG, "NULL argument");
    DeviceGuard dg(h);
    int rc;
    if (!h->pref_valid && (rc = launch_cfl_rate(h))) return rc;
    if ((rc = read_ctrl(h))) return rc;
    *p_ref = h->prec == KRATOS_PREC_MIXED ? h->h_ctrl->p_ref : 0.0;
    return KRATOS_OK;
}

int kratos_hydro_set_reference_pressure(kratos_hydro_t* h, double p_ref)
{
    if (!h) return fail(KRATOS_ERR_ARG, "NULL handle");
    const float m = (float)p_ref;   // the fp64 recovery and the fp32 solver must use the very same number
    if (!(m >= 0.0f) || !(m < 3.0e38f)) return fail(KRATOS_ERR_ARG, "reference pressure must be >= 0 and finite in fp32");
    DeviceGuard dg(h);
    {
        LaunchTimer lt(h, SLOT_OTHER);
        set_pref_kernel<<<1, 1, 0, h->stream>>>(h->ctrl, (double)m);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "set_reference_pressure: %s", cudaGetErrorString(e));
    h->pref_valid = true;
    return KRATOS_OK;
}

// ---------------------------------------------------------------------------------------
// kratos_hydro_totals_static: the conserved totals for a caller that may not allocate (see the header for who that is).
//
// kratos_hydro_totals needs a place for one double-double per field and thread block; a handle gets it from cudaMalloc.
// Here that place is part of the library image: a file-scope device array, present on every GPU the runtime has loaded
// this library onto, for as long as the process lives.  Layout: [5][592] dd partial sums, then 8 doubles of which the
// first 5 receive the finished totals when the caller wants them on the host.
//
// Host code must not hand `g_totals_static_scratch` itself to a kernel: in host code that name stands for a host-side
// shadow object, not for the array on the GPU.  The device address comes from cudaGetSymbolAddress, asked once per
// device with that device current, and is remembered in g_static_addr[].
#include <mutex>

namespace {

enum { STATIC_TOT_BLOCKS = 592, STATIC_TAIL_DOUBLES = 8, STATIC_MAX_DEVICES = 64 };
enum { STATIC_SCRATCH_DOUBLES = 2 * 5 * STATIC_TOT_BLOCKS + STATIC_TAIL_DOUBLES };
static_assert(sizeof(dd) == 2 * sizeof(double), "dd is two doubles");
static_assert(sizeof(double) * STATIC_SCRATCH_DOUBLES == KRATOS_TOTALS_STATIC_SCRATCH_BYTES, "header and array disagree");

static __device__ __align__(256) double g_totals_static_scratch[STATIC_SCRATCH_DOUBLES];

std::mutex g_static_mu;
double* g_static_addr[STATIC_MAX_DEVICES];  // device address of the array on device d; NULL = not asked yet

// Device address of the scratch array on the current device `dev` (first call per device: the look-up).
int static_scratch_on(int dev, double** out)
{
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(KRATOS_ERR_ARG, "totals_static: device ordinal %d not supported (< %d)", dev, (int)STATIC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_addr[dev]) {
        double* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_totals_static_scratch);
        if (e != cudaSuccess || !p)
            return fail(KRATOS_ERR_CUDA, "totals_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
        g_static_addr[dev] = p;
    }
    *out = g_static_addr[dev];
    return KRATOS_OK;
}

// true when p is device (or managed) memory that belongs to device dev
bool is_memory_of_device(const void* p, int dev)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) && a.device == dev;
}

}  // namespace

int kratos_hydro_totals_static(const double* U, long long ncell, double* out, int out_on_device, void* cuda_stream)
{
    if (!U || !out) return fail(KRATOS_ERR_ARG, "totals_static: NULL argument");
    if (ncell < 1 || ncell > KRATOS_TOTALS_STATIC_MAX_CELLS)
        return fail(KRATOS_ERR_ARG, "totals_static: ncell = %lld is outside 1 .. KRATOS_TOTALS_STATIC_MAX_CELLS = %lld",
                    ncell, (long long)KRATOS_TOTALS_STATIC_MAX_CELLS);
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (!is_memory_of_device(U, dev)) return fail(KRATOS_ERR_ARG, "totals_static: U is not device memory of the current device %d", dev);
    if (out_on_device && !is_memory_of_device(out, dev))
        return fail(KRATOS_ERR_ARG, "totals_static: out is not device memory of the current device %d (out_on_device = 1)", dev);
    double* scratch = nullptr;
    int rc = static_scratch_on(dev, &scratch);
    if (rc) return rc;

    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    // the grid of kratos_hydro_totals (kratos_hydro_create: tot_blocks), so that the sums come out in the same order
    const int blocks = (int)((ncell + 255) / 256 < STATIC_TOT_BLOCKS ? (ncell + 255) / 256 : STATIC_TOT_BLOCKS);
    dd* partial = reinterpret_cast<dd*>(scratch);
    double* tail = scratch + 2 * 5 * STATIC_TOT_BLOCKS;
    totals_kernel<double><<<dim3(blocks, 5), 256, 0, stream>>>(U, ncell, partial);
    totals_final_kernel<<<1, 32, 0, stream>>>(partial, blocks, out_on_device ? out : tail);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KRATOS_ERR_CUDA, "totals_static: launch: %s", cudaGetErrorString(e));
    if (!out_on_device) {
        CUDA_TRY(cudaMemcpyAsync(out, tail, sizeof(double) * 5, cudaMemcpyDeviceToHost, stream));
        CUDA_TRY(cudaStreamSynchronize(stream));
    }
    return KRATOS_OK;
}
