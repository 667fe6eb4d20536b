// hydro_api.cu -- the C-ABI of include/hydro.h over the sm_100a kernels.
// Host-side driver of Algorithm 1: persistent device state, one stream,
// no per-step host<->device traffic except the 8-byte max-signal-speed read when the host
// supplies dt (hydro_cfl_dt / hydro_evolve).
#include "../../include/hydro.h"
#include "hydro_kernels.cuh"
#include "hydro_stage_fused.cuh"
#include "hydro_stage_fused2d.cuh"
#include "hydro_stage_fused1d.cuh"
#include "hydro_stage_warp2d.cuh"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

using namespace hyd;

namespace {

thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};

void *(*g_alloc)(size_t, void *) = nullptr;
void (*g_release)(void *) = nullptr;

int fail(int code, const char *fmt, const char *a = "", const char *b = "")
{
    snprintf(g_err, sizeof g_err, fmt, a, b);
    return code;
}

#define CUDA_TRY(expr)                                                                   \
    do {                                                                                 \
        cudaError_t e_ = (expr);                                                         \
        if (e_ != cudaSuccess)                                                           \
            return fail(HYDRO_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_));        \
    } while (0)

#define LAUNCH_CHECK(name)                                                               \
    do {                                                                                 \
        g_launches.fetch_add(1, std::memory_order_relaxed);                              \
        cudaError_t e_ = cudaGetLastError();                                             \
        if (e_ != cudaSuccess)                                                           \
            return fail(HYDRO_ERR_CUDA, "launch %s: %s", name, cudaGetErrorString(e_));  \
    } while (0)

}  // namespace

struct hydro {
    Grid g;
    double dx, cfl;                 // dx = edge along x (dt/dx scales the update)
    double dxyz[3] = { 0, 0, 0 };   // cell edges; dmin = the smallest one over the active axes (R22)
    double dmin = 0.0;
    double *block = nullptr;        // one allocation: [A | B]
    double *A = nullptr, *B = nullptr;   // element (0,0,0) of variable 0 of each buffer
    size_t buf_doubles = 0;         // doubles per buffer incl. lead
    StepScalars *scal = nullptr;    // device scalars
    StepScalars *scal_host = nullptr;   // pinned mirror for small reads
    cudaStream_t stream = nullptr;
    bool own_alloc_default = true;  // allocated through cudaMalloc (vs the hook)
    void (*release)(void *) = nullptr;
    bool have_state = false;
    bool smax_valid = false;        // scal->smax_bits holds max(|v|+c) of the current state
    bool t_on_device = false;       // run_steps advanced the device clock
    bool ghosts_valid = false;      // periodic x / y ghost layers of A are current (fused kernel, variant 1)
    double t = 0.0;
    long long step = 0;
    int variant = 1;
    int w2rows = 0;                 // warp-column 2D kernel: rows per chunk (0: not chosen yet)
    AxisMap amap;                   // the caller's axes / variables -> internal ones (identity unless relabelled)
    bool relabelled = false;
    double *stage_io = nullptr;     // relabelled handle: device staging of hydro_set_state / hydro_get_state from / to host memory
    bool graph_replay = true;       // hydro_set_graph_replay
    int ty_req = 0, lz_req = 0;     // hydro_set_tiling (0 = chosen by the library)
    FusedPlan plan;                 // launch geometry / TMA descriptors of the fused kernel
    // one device-dt RK2 step (next_dt + stage launches) captured as a CUDA graph, replayed by
    // hydro_run_steps / hydro_evolve; rebuilt when anything baked into the launches changes
    cudaGraphExec_t step_graph = nullptr;
    int graph_kernels = 0;          // kernels per replay (for hydro_launch_count)
    // host mirror (hydro_host_alloc / hydro_update_device / hydro_update_host): pinned host buffers
    // owned by the handle, device staging buffers in the packed layout, one copy stream per direction
    std::vector<double *> host_bufs;
    double *stage_in = nullptr, *stage_out = nullptr;
    cudaStream_t cin = nullptr, cout = nullptr;
    cudaEvent_t ev_in_done = nullptr, ev_unpacked = nullptr, ev_packed = nullptr, ev_out_done = nullptr;
    // measurement hooks (hydro_set_profiling)
    bool profiling = false;
    struct Span { int which; cudaEvent_t a, b; };
    std::vector<Span> spans;
    std::vector<cudaEvent_t> pool;
};

namespace {

constexpr int LEAD = 14;            // doubles before (0,0,0): first active cell of a row is 128-B aligned

enum { K_GHOST = 0, K_STAGE1 = 1, K_STAGE2 = 2, K_NEXTDT = 3, K_CFL = 4 };

cudaEvent_t take_event(hydro *h)
{
    cudaEvent_t e = nullptr;
    if (!h->pool.empty()) { e = h->pool.back(); h->pool.pop_back(); return e; }
    if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return e;
}

// Brackets one kernel launch with events on the handle's stream while profiling is on.
struct Scope {
    hydro *h; int which; cudaEvent_t a = nullptr;
    Scope(hydro *h_, int w) : h(h_), which(w)
    {
        if (h->profiling && (a = take_event(h))) cudaEventRecord(a, h->stream);
    }
    ~Scope()
    {
        if (!a) return;                            // profiling off, or no event to be had: span dropped
        cudaEvent_t b = take_event(h);
        if (!b) { h->pool.push_back(a); return; }
        cudaEventRecord(b, h->stream);
        h->spans.push_back({which, a, b});
    }
};

int dev_alloc(hydro *h, void **p, size_t bytes)
{
    if (g_alloc) {
        *p = g_alloc(bytes, (void *)h->stream);
        h->own_alloc_default = false;
        h->release = g_release;
        return *p ? HYDRO_OK : fail(HYDRO_ERR_ALLOC, "allocator hook returned NULL%s%s");
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        *p = nullptr;
        return fail(HYDRO_ERR_ALLOC, "cudaMalloc: %s%s", cudaGetErrorString(e));
    }
    return HYDRO_OK;
}

void dev_free(hydro *h, void *p)
{
    if (!p) return;
    if (h->release) h->release(p);
    else cudaFree(p);
}

int is_device_pointer(const void *p, bool *on_device)
{
    cudaPointerAttributes a;
    cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) { cudaGetLastError(); *on_device = false; return HYDRO_OK; }
    *on_device = (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged);
    return HYDRO_OK;
}

// Boundaries of the fused stage kernels (variant 1; GhostExchange).  Outflow
// and reflecting rules are applied in the kernel and every z ghost plane is served by remapping the
// TMA plane coordinate, so only periodic x / y faces need ghost layers in memory.  Those are either
// kept current by the producer (wrap stores in the update; ghost_fill_kernel then runs once after the
// state was set from outside, ensure_ghosts) or filled by ghost_fill_kernel before every stage.  The
// first is one launch less per stage and wins up to 256^3 (64^3: 43 -> 39 us per step); on larger
// grids the partial-sector stores of the x images cost more than the fill kernel (512^3: stage 2
// +8 %), so those keep the fill.  Variant 2 (fused kernel, every ghost layer from memory) and the
// simple kernel fill all active axes before every stage.
int periodic_xy(const hydro *h)
{
    int axes = 0;
    if (h->g.bc[0] == HYDRO_BC_PERIODIC) axes |= 1;
    if (h->g.ndim >= 2 && h->g.bc[2] == HYDRO_BC_PERIODIC) axes |= 2;
    return axes;
}

bool fused_run(const hydro *h) { return h->variant == 1; }
bool warp2d_run(const hydro *h) { return h->g.ndim == 2 && h->variant == 3; }   // every boundary applied on the way in

int wrap_axes(const hydro *h)      // periodic axes whose ghost layers the stage kernels maintain
{
    const long long cells = (long long)h->g.nx * h->g.ny * h->g.nz;
    return fused_run(h) && h->g.ndim >= 2 && cells <= (1ll << 25) ? periodic_xy(h) : 0;
}

int fill_axes(const hydro *h)      // axes ghost_fill_kernel fills before every stage
{
    if (warp2d_run(h)) return 0;
    if (!fused_run(h)) return (1 << h->g.ndim) - 1;       // inactive axes have no ghost layers
    if (h->g.ndim == 1) return 0;                         // the 1D kernel reads source cells, wrap included
    return periodic_xy(h) & ~wrap_axes(h);
}

int inkernel_axes(const hydro *h)  // axes whose boundary rule the fused kernels apply themselves
{
    if (fused_run(h) && h->g.ndim == 1) return 1;
    return fused_run(h) ? ((1 << h->g.ndim) - 1) & ~periodic_xy(h) : 0;
}

int launch_ghost_fill(hydro *h, double *U, bool clear_smax, bool advance_dt = false, int axes = 7)
{
    const Grid &g = h->g;
    axes &= (1 << g.ndim) - 1;                               // inactive axes have no ghost layers
    const long long n = ((axes & 4) ? (long long)g.nx * g.ny : 0) + ((axes & 1) ? (long long)g.ny * g.nz : 0) +
                        ((axes & 2) ? (long long)g.nz * g.nx : 0);
    const int tb = 128;
    Scope sc(h, K_GHOST);
    ghost_fill_kernel<<<dim3((unsigned)((n + tb - 1) / tb), NVAR), tb, 0, h->stream>>>(
        g, U, clear_smax ? &h->scal->smax_bits : nullptr, advance_dt ? h->scal : nullptr,
        h->cfl / (double)g.ndim, h->dmin, axes);
    LAUNCH_CHECK("ghost_fill");
    return HYDRO_OK;
}

int launch_begin_step(hydro *h, bool advance_dt)
{
    Scope sc(h, K_NEXTDT);
    begin_step_kernel<<<1, 1, 0, h->stream>>>(h->scal, advance_dt ? 1 : 0, h->cfl / (double)h->g.ndim, h->dmin);
    LAUNCH_CHECK("begin_step");
    return HYDRO_OK;
}

int launch_cfl_reduce(hydro *h)
{
    CUDA_TRY(cudaMemsetAsync(&h->scal->smax_bits, 0, sizeof(unsigned long long), h->stream));
    const long long rows = (long long)h->g.ny * h->g.nz;
    long long blocks = (rows + 7) / 8;
    if (rows == 1) blocks = (h->g.nx + 255) / 256;          // 1D run: the warps of all blocks stride one row
    if (blocks > 148 * 8) blocks = 148 * 8;
    Scope sc(h, K_CFL);
    cfl_reduce_kernel<<<(unsigned)blocks, 256, 0, h->stream>>>(h->g, h->A, &h->scal->smax_bits,
                                                               &h->scal->flag);
    LAUNCH_CHECK("cfl_reduce");
    h->smax_valid = true;
    return HYDRO_OK;
}

// One substep over the active planes [kb, ke) (whole grid: 0, nz).
// After the state was set from outside, the periodic x / y ghost layers of A are filled once.
int ensure_ghosts(hydro *h)
{
    if (h->ghosts_valid) return HYDRO_OK;
    const int axes = wrap_axes(h);
    int rc;
    if (axes && (rc = launch_ghost_fill(h, h->A, false, false, axes))) return rc;
    h->ghosts_valid = true;
    return HYDRO_OK;
}

template <int STAGE>
int launch_stage(hydro *h, const double *in, const double *old, double *out, double r,
                 bool dev_dt, bool reduce, int kb = 0, int ke = -1)
{
    const Grid &g = h->g;
    if (ke < 0) ke = g.nz;
    if (ke <= kb) return HYDRO_OK;
    const StepScalars *dd = dev_dt ? h->scal : nullptr;
    StepScalars *red = reduce ? h->scal : nullptr;
    Scope sc(h, STAGE == 1 ? K_STAGE1 : K_STAGE2);
    if (h->variant == 0) {                    // (variants 1 and 2 are the fused kernels)
        dim3 tb(32, 4, 1);
        if (g.ndim == 1) tb = dim3(128, 1, 1);
        dim3 gr((g.nx + tb.x - 1) / tb.x, (g.ny + tb.y - 1) / tb.y, ke - kb);
        if (g.ndim == 1)      stage_simple_kernel<STAGE, 1><<<gr, tb, 0, h->stream>>>(g, in, old, out, r, dd, h->dx, red, kb);
        else if (g.ndim == 2) stage_simple_kernel<STAGE, 2><<<gr, tb, 0, h->stream>>>(g, in, old, out, r, dd, h->dx, red, kb);
        else                  stage_simple_kernel<STAGE, 3><<<gr, tb, 0, h->stream>>>(g, in, old, out, r, dd, h->dx, red, kb);
        LAUNCH_CHECK("stage_simple");
        return HYDRO_OK;
    }
    if (g.ndim == 1) {                        // fused 1D kernel
        cudaError_t e1 = launch_stage_fused1d<STAGE>(g, in, old, out, r, dd, h->dx, red, inkernel_axes(h) & 1, h->stream);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        if (e1 != cudaSuccess) return fail(HYDRO_ERR_CUDA, "launch stage_fused1d: %s%s", cudaGetErrorString(e1));
        return HYDRO_OK;
    }
    if (warp2d_run(h)) {                      // warp-column 2D kernel
        if (!h->w2rows) {
            int nsm = 148, dev = 0;
            if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
            h->w2rows = warp2d_choose_rows(g, nsm);
        }
        cudaError_t ew = launch_stage_warp2d<STAGE>(g, in, old, out, r, dd, h->dx, red, h->w2rows, h->stream);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        if (ew != cudaSuccess) return fail(HYDRO_ERR_CUDA, "launch stage_warp2d: %s%s", cudaGetErrorString(ew));
        return HYDRO_OK;
    }
    const int inbc = inkernel_axes(h);
    if (g.ndim == 2) {
        cudaError_t e2 = launch_stage_fused2d<STAGE>(h->plan, g, in, old, out, r, dd, h->dx, red, inbc, wrap_axes(h),
                                                     h->stream);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        if (e2 != cudaSuccess) return fail(HYDRO_ERR_CUDA, "launch stage_fused2d: %s%s", cudaGetErrorString(e2));
        return HYDRO_OK;
    }
    cudaError_t e = launch_stage_fused<STAGE>(h->plan, g, in, old, out, r, dd, h->dx, red, inbc, wrap_axes(h),
                                              h->stream, kb, ke);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (e != cudaSuccess) return fail(HYDRO_ERR_CUDA, "launch stage_fused: %s%s", cudaGetErrorString(e));
    return HYDRO_OK;
}

// One RK2 step (Algorithm 1 lines 6-21).  dt_host is ignored when dev_dt.
int enqueue_step(hydro *h, double dt_host, bool dev_dt)
{
    const double r = dt_host / h->dx;
    int rc;
    const int axes = fill_axes(h);
    if (axes) {
        // (simple kernel, variant 2) device dt: the first fill of the step also forms dt = (cfl/3) dx / smax and advances the
        // clock; the second one clears the accumulator of the reduction fused into stage 2
        if ((rc = launch_ghost_fill(h, h->A, false, dev_dt, axes))) return rc;
        if ((rc = launch_stage<1>(h, h->A, nullptr, h->B, r, dev_dt, false))) return rc;
        if ((rc = launch_ghost_fill(h, h->B, true, false, axes))) return rc;
    } else {
        // the stage kernels handle every boundary themselves: three launches per step
        if ((rc = launch_begin_step(h, dev_dt))) return rc;
        if ((rc = launch_stage<1>(h, h->A, nullptr, h->B, r, dev_dt, false))) return rc;
    }
    if ((rc = launch_stage<2>(h, h->B, h->A, h->A, r, dev_dt, true))) return rc;
    h->smax_valid = true;
    return HYDRO_OK;
}

int read_scalars(hydro *h)
{
    CUDA_TRY(cudaMemcpyAsync(h->scal_host, h->scal, sizeof(StepScalars), cudaMemcpyDeviceToHost,
                             h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (h->t_on_device) {
        h->t = h->scal_host->t;
        h->step += h->scal_host->steps;
        h->t_on_device = false;
    }
    return HYDRO_OK;
}

int copy_state(hydro *h, double *padded, double *packed, bool to_padded)
{
    const Grid &g = h->g;
    bool dev;
    is_device_pointer(packed, &dev);
    const long long nact = (long long)g.nx * g.ny * g.nz;
    long long blocks = (nact + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (!dev && h->relabelled) {
        // relabelled axes: a transposition is no pitched copy -- stage the packed state on the device
        const size_t bytes = (size_t)NVAR * nact * sizeof(double);
        if (!h->stage_io && cudaMalloc((void **)&h->stage_io, bytes) != cudaSuccess) {
            cudaGetLastError();
            return fail(HYDRO_ERR_ALLOC, "set/get_state: staging buffer%s%s");
        }
        if (to_padded) {
            CUDA_TRY(cudaMemcpyAsync(h->stage_io, packed, bytes, cudaMemcpyHostToDevice, h->stream));
            repack_kernel<true><<<(unsigned)blocks, 256, 0, h->stream>>>(g, h->amap, padded, h->stage_io, 31u);
            LAUNCH_CHECK("repack");
        } else {
            repack_kernel<false><<<(unsigned)blocks, 256, 0, h->stream>>>(g, h->amap, padded, h->stage_io, 31u);
            LAUNCH_CHECK("repack");
            CUDA_TRY(cudaMemcpyAsync(packed, h->stage_io, bytes, cudaMemcpyDeviceToHost, h->stream));
        }
        return HYDRO_OK;
    }
    if (dev) {
        if (to_padded) repack_kernel<true><<<(unsigned)blocks, 256, 0, h->stream>>>(g, h->amap, padded, packed, 31u);
        else repack_kernel<false><<<(unsigned)blocks, 256, 0, h->stream>>>(g, h->amap, padded, packed, 31u);
        LAUNCH_CHECK("repack");
        return HYDRO_OK;
    }
    // host pointer: one pitched 3-D copy per variable straight into / out of the padded interior
    for (int v = 0; v < NVAR; ++v) {
        cudaMemcpy3DParms p;
        memset(&p, 0, sizeof p);
        cudaPitchedPtr dp = make_cudaPitchedPtr(padded + v * g.sv, (size_t)g.px * sizeof(double),
                                                (size_t)g.px, (size_t)g.ny + 2 * g.oy);
        cudaPitchedPtr hp = make_cudaPitchedPtr(packed + (size_t)v * g.nx * g.ny * g.nz,
                                                (size_t)g.nx * sizeof(double), (size_t)g.nx,
                                                (size_t)g.ny);
        const cudaPos dpos = make_cudaPos(NG * sizeof(double), g.oy, g.oz);
        const cudaPos hpos = make_cudaPos(0, 0, 0);
        if (to_padded) { p.srcPtr = hp; p.srcPos = hpos; p.dstPtr = dp; p.dstPos = dpos; }
        else           { p.srcPtr = dp; p.srcPos = dpos; p.dstPtr = hp; p.dstPos = hpos; }
        p.extent = make_cudaExtent((size_t)g.nx * sizeof(double), (size_t)g.ny, (size_t)g.nz);
        p.kind = to_padded ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost;
        CUDA_TRY(cudaMemcpy3DAsync(&p, h->stream));
    }
    return HYDRO_OK;
}

void drop_graph(hydro *h)
{
    if (h->step_graph) { cudaGraphExecDestroy(h->step_graph); h->step_graph = nullptr; }
}

// n device-dt steps: replays of the captured one-step graph when possible (not on the legacy
// default stream, which cannot be captured, and not while per-kernel profiling is on).
int enqueue_device_steps(hydro *h, long long n)
{
    int rc;
    if ((rc = ensure_ghosts(h))) return rc;                  // not part of the captured step
    const bool use_graph = h->stream != nullptr && !h->profiling && h->graph_replay;
    if (use_graph && !h->step_graph) {
        const long long before = g_launches.load();
        cudaGraph_t graph = nullptr;
        CUDA_TRY(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
        rc = enqueue_step(h, 0.0, true);
        cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
        if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) return fail(HYDRO_ERR_CUDA, "graph capture: %s%s", cudaGetErrorString(e));
        e = cudaGraphInstantiate(&h->step_graph, graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) { h->step_graph = nullptr; return fail(HYDRO_ERR_CUDA, "graph instantiate: %s%s", cudaGetErrorString(e)); }
        h->graph_kernels = (int)(g_launches.load() - before);
        g_launches.store(before);                     // capture launched nothing
    }
    for (long long s = 0; s < n; ++s) {
        if (use_graph) {
            CUDA_TRY(cudaGraphLaunch(h->step_graph, h->stream));
            g_launches.fetch_add(h->graph_kernels, std::memory_order_relaxed);
        } else {
            if ((rc = enqueue_step(h, 0.0, true))) return rc;
        }
    }
    h->smax_valid = true;
    return HYDRO_OK;
}

int begin_run(hydro *h, double t_final)
{
    begin_run_kernel<<<1, 1, 0, h->stream>>>(h->scal, h->t, t_final);
    LAUNCH_CHECK("begin_run");
    h->t_on_device = true;
    return HYDRO_OK;
}

}  // namespace

extern "C" {

const char *hydro_last_error(void) { return g_err; }
long long hydro_launch_count(void) { return g_launches.load(); }

int hydro_is_verification_build(void)
{
#ifdef HYDRO_VERIFY
    return 1;
#else
    return 0;
#endif
}

int hydro_set_profiling(hydro_t *h, int enable)
{
    if (!h) return fail(HYDRO_ERR_ARG, "set_profiling: NULL handle%s%s");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (auto &s : h->spans) { h->pool.push_back(s.a); h->pool.push_back(s.b); }
    h->spans.clear();
    h->profiling = enable != 0;
    return HYDRO_OK;
}

int hydro_get_kernel_time(hydro_t *h, int which, double *ms, long long *count)
{
    if (!h || !ms || !count) return fail(HYDRO_ERR_ARG, "get_kernel_time: NULL argument%s%s");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    double total = 0.0;
    long long n = 0;
    for (auto &s : h->spans)
        if (s.which == which) {
            float t = 0.f;
            CUDA_TRY(cudaEventElapsedTime(&t, s.a, s.b));
            total += t;
            ++n;
        }
    *ms = total;
    *count = n;
    return HYDRO_OK;
}

int hydro_set_allocator(void *(*alloc)(size_t, void *), void (*release)(void *))
{
    if ((alloc == nullptr) != (release == nullptr))
        return fail(HYDRO_ERR_ARG, "set_allocator: pass both hooks or neither%s%s");
    g_alloc = alloc;
    g_release = release;
    return HYDRO_OK;
}

// Axis order.  The stage kernels tile x in units of 32 cells and y in units of 8 or 16 and march along z,
// so a 3D grid with one awkward extent (33 x 257 x 65: two 32-wide tile columns for 33 cells) is cheaper
// with its axes relabelled (257 x 65 x 33: measured 7.5 against 5.1 G cell-updates/s).  The scheme is
// symmetric under relabelling -- exactly so in the oracle's association (pins P4, P10), to roundoff in the
// production arithmetic -- so the library may hold such a run relabelled: the launch-geometry cost model is
// evaluated for the six orders and another order is taken when it is at least 12 % cheaper.  Only the
// copies in and out of the handle know (AxisMap); cubic cells, no slab interface, 2^15 cells and more.
static void choose_axis_order(const int n[3], int nsm, int ax[3])
{
    static const int perms[6][3] = { { 0, 1, 2 }, { 0, 2, 1 }, { 1, 0, 2 }, { 1, 2, 0 }, { 2, 0, 1 }, { 2, 1, 0 } };
    double best = 1e300, ident = 0.0;
    int bi = 0;
    for (int p = 0; p < 6; ++p) {
        Grid t{};
        int e[3];
        for (int a = 0; a < 3; ++a) e[perms[p][a]] = n[a];
        t.nx = e[0]; t.ny = e[1]; t.nz = e[2];
        const double c16 = fused_partition(t, 16, 0, t.nz, nsm, 0).cost, c8 = fused_partition(t, 8, 0, t.nz, nsm, 0).cost;
        const double c = c16 < c8 ? c16 : c8;
        if (p == 0) ident = c;
        if (c < best - 1e-9) { best = c; bi = p; }
    }
    if (best > 0.88 * ident) bi = 0;
    for (int a = 0; a < 3; ++a) ax[a] = perms[bi][a];
}

static int create_nd(int ndim, const int n_user[3], const double d[3], double gamma, const int bc_user[6],
                     bool may_relabel, hydro_t **out);

int hydro_create_nd(int ndim, const int n[3], const double d[3], double gamma, const int bc[6],
                    hydro_t **out)
{
    return create_nd(ndim, n, d, gamma, bc, true, out);
}

static int create_nd(int ndim, const int n[3], const double d[3], double gamma, const int bc[6],
                     bool may_relabel, hydro_t **out)
{
    if (!out) return fail(HYDRO_ERR_ARG, "create: out is NULL%s%s");
    *out = nullptr;
    if (!bc || !n || !d) return fail(HYDRO_ERR_ARG, "create: NULL argument%s%s");
    if (ndim < 1 || ndim > 3) return fail(HYDRO_ERR_ARG, "create: ndim must be 1, 2 or 3%s%s");
    if (!(gamma > 1.0) || !std::isfinite(gamma)) return fail(HYDRO_ERR_ARG, "create: gamma must be > 1%s%s");
    for (int a = 0; a < 3; ++a) {
        if (a < ndim) {
            if (n[a] < 2) return fail(HYDRO_ERR_ARG, "create: an active axis needs >= 2 cells%s%s");
            if (!(d[a] > 0.0) || !std::isfinite(d[a])) return fail(HYDRO_ERR_ARG, "create: cell edges must be > 0%s%s");
            const int kmax = a == 2 ? HYDRO_BC_NEIGHBOUR : HYDRO_BC_PERIODIC;   // slabs are cut along z
            if (bc[2 * a] < 0 || bc[2 * a] > kmax || bc[2 * a + 1] < 0 || bc[2 * a + 1] > kmax)
                return fail(HYDRO_ERR_ARG, "create: unknown boundary kind%s%s");
            if ((bc[2 * a] == HYDRO_BC_PERIODIC) != (bc[2 * a + 1] == HYDRO_BC_PERIODIC))
                return fail(HYDRO_ERR_ARG, "create: periodic must be set on both faces of an axis%s%s");
        } else if (n[a] != 1) {
            return fail(HYDRO_ERR_ARG, "create: an inactive axis must have exactly one cell%s%s");
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(HYDRO_ERR_CUDA, "create: no CUDA device (there is no CPU fallback)%s%s");
    }
    hydro *h = new (std::nothrow) hydro;
    if (!h) return fail(HYDRO_ERR_ALLOC, "create: host allocation failed%s%s");
    // axis order: identity unless a relabelled order is clearly cheaper (see choose_axis_order)
    int ax[3] = { 0, 1, 2 };
    bool slab_face = false;
    for (int f = 0; f < 6; ++f) slab_face = slab_face || bc[f] == HYDRO_BC_NEIGHBOUR;
    if (may_relabel && ndim == 3 && !slab_face && d[0] == d[1] && d[1] == d[2] &&
        (long long)n[0] * n[1] * n[2] >= (1ll << 15)) {
        int nsm = 148, dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        choose_axis_order(n, nsm, ax);
    }
    h->relabelled = ax[0] != 0 || ax[1] != 1;
    int n_int[3], bc_int[6];
    for (int a = 0; a < 3; ++a) {
        h->amap.n[a] = n[a]; h->amap.ax[a] = ax[a]; h->amap.var[1 + a] = 1 + ax[a];
        n_int[ax[a]] = n[a]; bc_int[2 * ax[a]] = bc[2 * a]; bc_int[2 * ax[a] + 1] = bc[2 * a + 1];
    }
    h->amap.var[0] = 0; h->amap.var[4] = 4;
    n = n_int; bc = bc_int;                               // from here on: the internal axes
    const int nx = n[0], ny = n[1], nz = n[2];
    Grid &g = h->g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.ndim = ndim; g.oy = ndim >= 2 ? NG : 0; g.oz = ndim >= 3 ? NG : 0;
    g.px = ((nx + 2 * NG + 15) / 16) * 16;
    g.sy = (long long)g.px * (ny + 2 * g.oy);
    const long long vol = g.sy * (nz + 2 * g.oz);
    g.sv = ((vol + 15) / 16) * 16;
    for (int f = 0; f < 6; ++f) g.bc[f] = f < 2 * ndim ? bc[f] : HYDRO_BC_OUTFLOW;
    g.gamma = gamma; g.gm1 = gamma - 1.0; g.igm1 = 1.0 / g.gm1; g.theta = 1.4;
    h->dx = d[0]; h->cfl = 0.7;
    // 2D runs of a megacell and more default to the warp-column kernel (never slower there, 10-15 % faster
    // around 1024^2 - 2048^2; smaller grids are better off with the tiled kernel: DESIGN.md section 6.4)
    if (ndim == 2 && (long long)n[0] * n[1] >= (1ll << 20)) h->variant = 3;
    h->dmin = d[0];
    for (int a = 0; a < 3; ++a) {
        h->dxyz[a] = a < ndim ? d[a] : d[0];
        if (a < ndim && d[a] < h->dmin) h->dmin = d[a];
    }
    g.ry = h->dx / h->dxyz[1]; g.rz = h->dx / h->dxyz[2];
    // +16 tail so vectorised / TMA reads that run a few doubles past the last row stay inside
    h->buf_doubles = (size_t)LEAD + (size_t)NVAR * g.sv + 16 + 2;
    h->buf_doubles = ((h->buf_doubles + 15) / 16) * 16;
    void *p = nullptr;
    int rc = dev_alloc(h, &p, 2 * h->buf_doubles * sizeof(double));
    if (rc) { delete h; return rc; }
    h->block = (double *)p;
    h->A = h->block + LEAD;
    h->B = h->block + h->buf_doubles + LEAD;
    cudaError_t e = cudaMalloc((void **)&h->scal, sizeof(StepScalars));
    if (e == cudaSuccess) e = cudaMallocHost((void **)&h->scal_host, sizeof(StepScalars));
    if (e == cudaSuccess) e = cudaMemset(h->block, 0, 2 * h->buf_doubles * sizeof(double));
    if (e == cudaSuccess) e = cudaMemset(h->scal, 0, sizeof(StepScalars));
    if (e == cudaSuccess && ndim == 3) e = plan_stage_fused(h->plan, g, h->A, h->B);
    if (e == cudaSuccess && ndim == 2) e = plan_stage_fused2d(h->plan, g, h->A, h->B);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();   // the memsets ran on the legacy stream; the handle's
                                                         // stream may be a non-blocking one
    if (e != cudaSuccess) {
        cudaGetLastError();
        fail(HYDRO_ERR_CUDA, "create: %s%s", cudaGetErrorString(e));
        hydro_destroy(h);
        return HYDRO_ERR_CUDA;
    }
    *out = h;
    return HYDRO_OK;
}

int hydro_create(int nx, int ny, int nz, double gamma, double dx, const int bc[6], hydro_t **out)
{
    if (out) *out = nullptr;
    if (nx < 2 || ny < 2 || nz < 2) return fail(HYDRO_ERR_ARG, "create: nx,ny,nz must be >= 2%s%s");
    if (!(dx > 0.0) || !std::isfinite(dx)) return fail(HYDRO_ERR_ARG, "create: dx must be > 0%s%s");
    const int n[3] = { nx, ny, nz };
    const double d[3] = { dx, dx, dx };
    return hydro_create_nd(3, n, d, gamma, bc, out);
}

int hydro_destroy(hydro_t *h)
{
    if (!h) return fail(HYDRO_ERR_ARG, "destroy: NULL handle%s%s");
    cudaStreamSynchronize(h->stream);
    drop_graph(h);
    for (auto &s : h->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
    for (auto e : h->pool) cudaEventDestroy(e);
    if (h->cin) { cudaStreamSynchronize(h->cin); cudaStreamDestroy(h->cin); }
    if (h->cout) { cudaStreamSynchronize(h->cout); cudaStreamDestroy(h->cout); }
    for (cudaEvent_t e : { h->ev_in_done, h->ev_unpacked, h->ev_packed, h->ev_out_done })
        if (e) cudaEventDestroy(e);
    for (double *p : h->host_bufs) cudaFreeHost(p);
    if (h->stage_in) cudaFree(h->stage_in);
    if (h->stage_out) cudaFree(h->stage_out);
    if (h->stage_io) cudaFree(h->stage_io);
    dev_free(h, h->block);
    if (h->scal) cudaFree(h->scal);
    if (h->scal_host) cudaFreeHost(h->scal_host);
    delete h;
    return HYDRO_OK;
}

int hydro_set_stream(hydro_t *h, void *s)
{
    if (!h) return fail(HYDRO_ERR_ARG, "set_stream: NULL handle%s%s");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    drop_graph(h);
    h->stream = (cudaStream_t)s;
    return HYDRO_OK;
}

int hydro_set_cfl(hydro_t *h, double cfl)
{
    if (!h || !(cfl > 0.0) || !std::isfinite(cfl)) return fail(HYDRO_ERR_ARG, "set_cfl: cfl must be > 0%s%s");
    h->cfl = cfl;
    drop_graph(h);
    return HYDRO_OK;
}

int hydro_set_limiter_theta(hydro_t *h, double theta)
{
    if (!h || !(theta >= 1.0 && theta <= 2.0))
        return fail(HYDRO_ERR_ARG, "set_limiter_theta: theta must be in [1,2]%s%s");
    h->g.theta = theta;
    drop_graph(h);
    return HYDRO_OK;
}

int hydro_set_kernel_variant(hydro_t *h, int variant)
{
    if (!h || variant < 0 || variant > 3) return fail(HYDRO_ERR_ARG, "set_kernel_variant: 0, 1, 2 or 3%s%s");
    if (variant == 3 && h->g.ndim != 2)
        return fail(HYDRO_ERR_ARG, "set_kernel_variant: variant 3 is the warp-column kernel of 2D runs%s%s");
    if (h->g.ndim == 1 && variant == 2)
        return fail(HYDRO_ERR_ARG, "set_kernel_variant: a 1D run has variants 0 and 1%s%s");
    h->variant = variant;
    h->ghosts_valid = false;
    drop_graph(h);
    return HYDRO_OK;
}

int hydro_set_graph_replay(hydro_t *h, int enable)
{
    if (!h) return fail(HYDRO_ERR_ARG, "set_graph_replay: NULL handle%s%s");
    h->graph_replay = enable != 0;
    if (!h->graph_replay) { CUDA_TRY(cudaStreamSynchronize(h->stream)); drop_graph(h); }
    return HYDRO_OK;
}

int hydro_set_tiling(hydro_t *h, int tile_rows, int planes_per_chunk)
{
    if (!h) return fail(HYDRO_ERR_ARG, "set_tiling: NULL handle%s%s");
    if ((tile_rows != 0 && tile_rows != 8 && tile_rows != 16) || planes_per_chunk < 0)
        return fail(HYDRO_ERR_ARG, "set_tiling: tile_rows must be 0, 8 or 16 and planes_per_chunk >= 0%s%s");
    if (h->g.ndim == 1 || (h->g.ndim == 2 && tile_rows == 8))
        return fail(HYDRO_ERR_ARG, "set_tiling: 1D runs have no fused kernel; 2D runs use 32 x 16 tiles%s%s");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    drop_graph(h);
    h->ty_req = tile_rows; h->lz_req = planes_per_chunk;
    cudaError_t e = h->g.ndim == 2 ? plan_stage_fused2d(h->plan, h->g, h->A, h->B, h->lz_req)
                                   : plan_stage_fused(h->plan, h->g, h->A, h->B, h->ty_req, h->lz_req);
    if (e != cudaSuccess) return fail(HYDRO_ERR_CUDA, "set_tiling: %s%s", cudaGetErrorString(e));
    return HYDRO_OK;
}

int hydro_get_tiling(hydro_t *h, int *tile_rows, int *planes_per_chunk, long long *blocks)
{
    if (!h) return fail(HYDRO_ERR_ARG, "get_tiling: NULL handle%s%s");
    if (tile_rows) *tile_rows = h->plan.ty;
    if (planes_per_chunk) *planes_per_chunk = h->plan.lz;
    if (blocks) *blocks = (long long)h->plan.grid.x * h->plan.grid.y * h->plan.grid.z;
    return HYDRO_OK;
}

int hydro_tiling_partition(int nx, int ny, int nz, int tile_rows, int planes_per_chunk, int sms, int kb, int ke,
                           int out[5])
{
    if (nx < 1 || ny < 1 || nz < 1 || (tile_rows != 8 && tile_rows != 16) || planes_per_chunk < 0 || sms < 1 ||
        kb < 0 || ke > nz || ke <= kb || !out)
        return fail(HYDRO_ERR_ARG, "tiling_partition: bad argument%s%s");
    Grid g{};
    g.nx = nx; g.ny = ny; g.nz = nz;
    const FusedLayers z = fused_partition(g, tile_rows, kb, ke, sms, planes_per_chunk);
    out[0] = z.lz; out[1] = z.km; out[2] = z.nprim; out[3] = z.lzr; out[4] = z.nlayer;
    return HYDRO_OK;
}

int hydro_get_axis_order(hydro_t *h, int order[3])
{
    if (!h || !order) return fail(HYDRO_ERR_ARG, "get_axis_order: NULL argument%s%s");
    for (int a = 0; a < 3; ++a) order[a] = h->amap.ax[a];
    return HYDRO_OK;
}

int hydro_set_state(hydro_t *h, const double *U)
{
    if (!h || !U) return fail(HYDRO_ERR_ARG, "set_state: NULL argument%s%s");
    int rc = copy_state(h, h->A, const_cast<double *>(U), true);
    if (rc) return rc;
    CUDA_TRY(cudaMemsetAsync(h->scal, 0, sizeof(StepScalars), h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));   // host or device pointer: the caller may free or
                                                  // overwrite U on return (hydro.h)
    h->t = 0.0; h->step = 0; h->have_state = true; h->smax_valid = false; h->t_on_device = false;
    h->ghosts_valid = false;
    return HYDRO_OK;
}

int hydro_get_state(hydro_t *h, double *U)
{
    if (!h || !U) return fail(HYDRO_ERR_ARG, "get_state: NULL argument%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "get_state before set_state%s%s");
    int rc = copy_state(h, h->A, U, false);
    if (rc) return rc;
    if ((rc = read_scalars(h))) return rc;
    if (h->scal_host->flag) return fail(HYDRO_ERR_UNPHYSICAL, "unphysical state (rho<=0, p<=0 or non-finite speed)%s%s");
    return HYDRO_OK;
}

int hydro_ghost_fill(hydro_t *h)
{
    if (!h) return fail(HYDRO_ERR_ARG, "ghost_fill: NULL handle%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "ghost_fill before set_state%s%s");
    return launch_ghost_fill(h, h->A, false);
}

int hydro_get_padded(hydro_t *h, double *Upad)
{
    if (!h || !Upad) return fail(HYDRO_ERR_ARG, "get_padded: NULL argument%s%s");
    if (h->relabelled) return fail(HYDRO_ERR_ARG, "get_padded: the handle holds its axes relabelled (hydro_get_axis_order)%s%s");
    const Grid &g = h->g;
    const size_t Nx = g.nx + 2 * NG, Ny = g.ny + 2 * g.oy, Nz = g.nz + 2 * g.oz;
    for (int v = 0; v < NVAR; ++v)
        for (size_t K = 0; K < Nz; ++K)
            CUDA_TRY(cudaMemcpy2DAsync(Upad + ((size_t)v * Nz + K) * Ny * Nx, Nx * sizeof(double),
                                       h->A + v * g.sv + K * g.sy, (size_t)g.px * sizeof(double),
                                       Nx * sizeof(double), Ny, cudaMemcpyDefault, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return HYDRO_OK;
}

int hydro_max_signal_speed(hydro_t *h, double *smax)
{
    if (!h || !smax) return fail(HYDRO_ERR_ARG, "max_signal_speed: NULL argument%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "max_signal_speed before set_state%s%s");
    int rc;
    if (!h->smax_valid && (rc = launch_cfl_reduce(h))) return rc;
    if ((rc = read_scalars(h))) return rc;
    double s;
    memcpy(&s, &h->scal_host->smax_bits, sizeof s);
    *smax = s;
    if (h->scal_host->flag) return fail(HYDRO_ERR_UNPHYSICAL, "unphysical state (rho<=0, p<=0 or non-finite speed)%s%s");
    return HYDRO_OK;
}

int hydro_cfl_dt(hydro_t *h, double *dt)
{
    if (!dt) return fail(HYDRO_ERR_ARG, "cfl_dt: NULL argument%s%s");
    double smax;
    int rc = hydro_max_signal_speed(h, &smax);
    if (rc) return rc;
    const double c3 = h->cfl / (double)h->g.ndim;
    const double dxs = h->dmin / smax;
    *dt = c3 * dxs;
    return HYDRO_OK;
}

int hydro_step(hydro_t *h, double dt)
{
    if (!h) return fail(HYDRO_ERR_ARG, "step: NULL handle%s%s");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(HYDRO_ERR_ARG, "step: dt must be > 0 and finite%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "step before set_state%s%s");
    int rc;
    if (h->t_on_device && (rc = read_scalars(h))) return rc;
    if ((rc = ensure_ghosts(h))) return rc;
    if ((rc = enqueue_step(h, dt, false))) return rc;
    h->t = h->t + dt;
    h->step += 1;
    return HYDRO_OK;
}

int hydro_run_steps(hydro_t *h, long long n)
{
    if (!h || n < 0) return fail(HYDRO_ERR_ARG, "run_steps: bad argument%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "run_steps before set_state%s%s");
    if (n == 0) return HYDRO_OK;
    int rc;
    if (!h->smax_valid && (rc = launch_cfl_reduce(h))) return rc;
    if (!h->t_on_device && (rc = begin_run(h, HUGE_VAL))) return rc;
    return enqueue_device_steps(h, n);
}

// Algorithm 1's while loop with the time step kept on the device: batches of steps are enqueued
// without a host round trip; the kernel that forms dt clips the last step onto t_final and turns
// any step enqueued beyond it into the identity, so the host only reads the scalars once per batch.
int hydro_evolve(hydro_t *h, double t_final, long long *nsteps)
{
    if (!h || !std::isfinite(t_final)) return fail(HYDRO_ERR_ARG, "evolve: bad argument%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "evolve before set_state%s%s");
    int rc;
    if (h->t_on_device && (rc = read_scalars(h))) return rc;
    if (t_final < h->t) return fail(HYDRO_ERR_ARG, "evolve: t_final is in the past%s%s");
    if (nsteps) *nsteps = 0;
    if (!(h->t < t_final)) return HYDRO_OK;
    if (!h->smax_valid && (rc = launch_cfl_reduce(h))) return rc;
    if ((rc = begin_run(h, t_final))) return rc;
    long long batch = 4;
    double t_prev = h->t;
    for (;;) {
        if ((rc = enqueue_device_steps(h, batch))) return rc;
        CUDA_TRY(cudaMemcpyAsync(h->scal_host, h->scal, sizeof(StepScalars), cudaMemcpyDeviceToHost,
                                 h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        const StepScalars &sc = *h->scal_host;
        if (sc.flag) {
            h->t = sc.t; h->step += sc.steps; h->t_on_device = false;
            return fail(HYDRO_ERR_UNPHYSICAL, "unphysical state (rho<=0, p<=0 or non-finite speed)%s%s");
        }
        if (sc.done) break;
        // no progress (dt underflowed to 0, or the signal speed is so large that t + dt == t):
        // bail out instead of looping forever
        if (!(sc.dt > 0.0) || !(sc.t > t_prev)) {
            h->t = sc.t; h->step += sc.steps; h->t_on_device = false;
            return fail(HYDRO_ERR_UNPHYSICAL, "evolve: the time step no longer advances the clock%s%s");
        }
        t_prev = sc.t;
        // size the next batch from the time left and the last dt (wasted identity steps are cheap
        // but not free); never more than 64 steps between host checks
        const double left = (t_final - sc.t) / (sc.dt > 0.0 ? sc.dt : 1.0);
        batch = left < 1.0 ? 1 : (left > 64.0 ? 64 : (long long)left + 1);
    }
    h->t = h->scal_host->t;                       // == t_final exactly
    h->step += h->scal_host->steps;
    h->t_on_device = false;
    if (nsteps) *nsteps = h->scal_host->steps;
    return HYDRO_OK;
}

// ---- host mirror (the paper's StorageForm: PAPER.md:62, 359-363) ----

namespace {
int mirror_setup(hydro *h)
{
    if (h->cin) return HYDRO_OK;
    CUDA_TRY(cudaStreamCreateWithFlags(&h->cin, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&h->cout, cudaStreamNonBlocking));
    for (cudaEvent_t *e : { &h->ev_in_done, &h->ev_unpacked, &h->ev_packed, &h->ev_out_done })
        CUDA_TRY(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    return HYDRO_OK;
}
size_t packed_doubles(const hydro *h) { return (size_t)NVAR * h->g.nx * h->g.ny * h->g.nz; }
// copies the selected fields (runs of adjacent fields as one transfer)
int copy_fields(double *dst, const double *src, size_t n, unsigned fields, cudaMemcpyKind kind, cudaStream_t st)
{
    for (int v = 0; v < NVAR;) {
        if (!(fields >> v & 1u)) { ++v; continue; }
        int w = v;
        while (w + 1 < NVAR && (fields >> (w + 1) & 1u)) ++w;
        CUDA_TRY(cudaMemcpyAsync(dst + v * n, src + v * n, (size_t)(w - v + 1) * n * sizeof(double), kind, st));
        v = w + 1;
    }
    return HYDRO_OK;
}
unsigned repack_blocks(const hydro *h)
{
    const long long nact = (long long)h->g.nx * h->g.ny * h->g.nz;
    long long b = (nact + 255) / 256;
    return (unsigned)(b > 148 * 16 ? 148 * 16 : b);
}
}  // namespace

int hydro_host_alloc(hydro_t *h, double **U_host)
{
    if (!h || !U_host) return fail(HYDRO_ERR_ARG, "host_alloc: NULL argument%s%s");
    double *p = nullptr;
    cudaError_t e = cudaHostAlloc((void **)&p, packed_doubles(h) * sizeof(double), cudaHostAllocDefault);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(HYDRO_ERR_ALLOC, "host_alloc: %s%s", cudaGetErrorString(e)); }
    h->host_bufs.push_back(p);
    *U_host = p;
    return HYDRO_OK;
}

int hydro_update_device(hydro_t *h, unsigned fields, const double *U_host)
{
    if (!h || !U_host || !(fields & 31u) || (fields & ~31u)) return fail(HYDRO_ERR_ARG, "update_device: bad argument%s%s");
    if (!h->have_state && (fields & 31u) != 31u)
        return fail(HYDRO_ERR_NOSTATE, "update_device: the first update must bring all five fields%s%s");
    int rc = mirror_setup(h);
    if (rc) return rc;
    const size_t n = (size_t)h->g.nx * h->g.ny * h->g.nz;
    if (!h->stage_in) {
        cudaError_t e = cudaMalloc((void **)&h->stage_in, NVAR * n * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); return fail(HYDRO_ERR_ALLOC, "update_device: %s%s", cudaGetErrorString(e)); }
        CUDA_TRY(cudaEventRecord(h->ev_unpacked, h->stream));
    }
    // copy stream: after the previous unpack has read the staging buffer; then H2D of the selected fields
    CUDA_TRY(cudaStreamWaitEvent(h->cin, h->ev_unpacked, 0));
    if ((rc = copy_fields(h->stage_in, U_host, n, fields, cudaMemcpyHostToDevice, h->cin))) return rc;
    CUDA_TRY(cudaEventRecord(h->ev_in_done, h->cin));
    // compute stream: whatever was enqueued before keeps running during the transfer; the unpack
    // (and everything enqueued after this call) waits for it
    CUDA_TRY(cudaStreamWaitEvent(h->stream, h->ev_in_done, 0));
    if (h->t_on_device && (rc = read_scalars(h))) return rc;
    repack_kernel<true><<<repack_blocks(h), 256, 0, h->stream>>>(h->g, h->amap, h->A, h->stage_in, fields);
    LAUNCH_CHECK("unpack");
    CUDA_TRY(cudaEventRecord(h->ev_unpacked, h->stream));
    CUDA_TRY(cudaMemsetAsync(&h->scal->flag, 0, sizeof(int), h->stream));
    h->have_state = true; h->smax_valid = false; h->ghosts_valid = false;
    return HYDRO_OK;
}

int hydro_update_host(hydro_t *h, unsigned fields, double *U_host)
{
    if (!h || !U_host || !(fields & 31u) || (fields & ~31u)) return fail(HYDRO_ERR_ARG, "update_host: bad argument%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "update_host before any state%s%s");
    int rc = mirror_setup(h);
    if (rc) return rc;
    const size_t n = (size_t)h->g.nx * h->g.ny * h->g.nz;
    if (!h->stage_out) {
        cudaError_t e = cudaMalloc((void **)&h->stage_out, NVAR * n * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); return fail(HYDRO_ERR_ALLOC, "update_host: %s%s", cudaGetErrorString(e)); }
        CUDA_TRY(cudaEventRecord(h->ev_out_done, h->cout));
    }
    // compute stream: snapshot of the selected fields into the packed staging buffer (HBM to HBM), after
    // the previous device-to-host transfer has drained it; the steps enqueued next do not wait
    CUDA_TRY(cudaStreamWaitEvent(h->stream, h->ev_out_done, 0));
    repack_kernel<false><<<repack_blocks(h), 256, 0, h->stream>>>(h->g, h->amap, h->A, h->stage_out, fields);
    LAUNCH_CHECK("pack");
    CUDA_TRY(cudaEventRecord(h->ev_packed, h->stream));
    CUDA_TRY(cudaStreamWaitEvent(h->cout, h->ev_packed, 0));
    if ((rc = copy_fields(U_host, h->stage_out, n, fields, cudaMemcpyDeviceToHost, h->cout))) return rc;
    CUDA_TRY(cudaEventRecord(h->ev_out_done, h->cout));
    return HYDRO_OK;
}

int hydro_transfer_sync(hydro_t *h)
{
    if (!h) return fail(HYDRO_ERR_ARG, "transfer_sync: NULL handle%s%s");
    if (h->cin) CUDA_TRY(cudaStreamSynchronize(h->cin));
    if (h->cout) CUDA_TRY(cudaStreamSynchronize(h->cout));
    return HYDRO_OK;
}

// ---- slab decomposition along z ------------------------

int hydro_create_slab(int nx, int ny, int nz_global, double gamma, double dx, const int bc[6],
                      int rank, int nranks, hydro_t **out, int *k_first, int *nz_local)
{
    if (out) *out = nullptr;
    if (!out || !bc) return fail(HYDRO_ERR_ARG, "create_slab: NULL argument%s%s");
    if (nranks < 1 || rank < 0 || rank >= nranks) return fail(HYDRO_ERR_ARG, "create_slab: bad rank%s%s");
    if (nz_global < 2 * nranks) return fail(HYDRO_ERR_ARG, "create_slab: every slab needs >= 2 planes%s%s");
    for (int f = 0; f < 6; ++f)
        if (bc[f] < 0 || bc[f] > 2) return fail(HYDRO_ERR_ARG, "create_slab: unknown boundary kind%s%s");
    // planes [k0, k0 + nzl): the first nz_global % nranks slabs get one plane more
    const int base = nz_global / nranks, extra = nz_global % nranks;
    const int nzl = base + (rank < extra ? 1 : 0);
    const int k0 = rank * base + (rank < extra ? rank : extra);
    int b[6];
    memcpy(b, bc, sizeof b);
    const bool periodic_z = bc[4] == HYDRO_BC_PERIODIC;
    if (nranks > 1) {
        if (rank > 0 || periodic_z) b[4] = HYDRO_BC_NEIGHBOUR;
        if (rank < nranks - 1 || periodic_z) b[5] = HYDRO_BC_NEIGHBOUR;
    }
    if (k_first) *k_first = k0;
    if (nz_local) *nz_local = nzl;
    if (nx < 2 || ny < 2) return fail(HYDRO_ERR_ARG, "create_slab: nx,ny must be >= 2%s%s");
    const int n[3] = { nx, ny, nzl };
    const double d[3] = { dx, dx, dx };
    return create_nd(3, n, d, gamma, b, false, out);
}

int hydro_halo_count(hydro_t *h, size_t *doubles)
{
    if (!h || !doubles) return fail(HYDRO_ERR_ARG, "halo_count: NULL argument%s%s");
    *doubles = (size_t)NVAR * 2 * h->g.ny * h->g.nx;
    return HYDRO_OK;
}

namespace {
int halo_blocks(const hydro *h)
{
    const long long total = 10ll * h->g.ny * h->g.nx;
    long long b = (total + 255) / 256;
    return (int)(b > 148 * 8 ? 148 * 8 : b);
}
int halo_args(hydro *h, int which, int side, const void *p, const char *who)
{
    if (!h || !p || (which != 0 && which != 1) || (side != 0 && side != 1))
        return fail(HYDRO_ERR_ARG, "%s: bad argument%s", who);
    if (h->g.ndim != 3) return fail(HYDRO_ERR_ARG, "%s: slabs are cut along z of a 3D run%s", who);
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "%s before set_state%s", who);
    return HYDRO_OK;
}
}  // namespace

int hydro_halo_pack(hydro_t *h, int which, int side, double *dst)
{
    int rc = halo_args(h, which, side, dst, "halo_pack");
    if (rc) return rc;
    const Grid &g = h->g;
    halo_kernel<0><<<halo_blocks(h), 256, 0, h->stream>>>(g, which ? h->B : h->A, dst, side ? g.nz : NG, 0, 0);
    LAUNCH_CHECK("halo_pack");
    return HYDRO_OK;
}

int hydro_halo_unpack(hydro_t *h, int which, int side, const double *src)
{
    int rc = halo_args(h, which, side, src, "halo_unpack");
    if (rc) return rc;
    const Grid &g = h->g;
    halo_kernel<1><<<halo_blocks(h), 256, 0, h->stream>>>(g, which ? h->B : h->A, const_cast<double *>(src),
                                                          side ? g.nz + NG : 0, 0, 0);
    LAUNCH_CHECK("halo_unpack");
    return HYDRO_OK;
}

int hydro_state_base(hydro_t *h, int which, double **base, int *nz_local, long long *var_stride)
{
    if (!h || !base || (which != 0 && which != 1)) return fail(HYDRO_ERR_ARG, "state_base: bad argument%s%s");
    *base = which ? h->B : h->A;
    if (nz_local) *nz_local = h->g.nz;
    if (var_stride) *var_stride = h->g.sv;
    return HYDRO_OK;
}

int hydro_halo_push(hydro_t *h, int which, int side, double *peer_base, int peer_nz, long long peer_var_stride)
{
    int rc = halo_args(h, which, side, peer_base, "halo_push");
    if (rc) return rc;
    const Grid &g = h->g;
    // my low boundary planes fill the neighbour's HIGH ghost planes and vice versa
    const int K0 = side ? g.nz : NG, Kd = side ? 0 : peer_nz + NG;
    halo_kernel<2><<<halo_blocks(h), 256, 0, h->stream>>>(g, which ? h->B : h->A, peer_base, K0, Kd, peer_var_stride);
    LAUNCH_CHECK("halo_push");
    return HYDRO_OK;
}

int hydro_smax_device(hydro_t *h, double **smax)
{
    if (!h || !smax) return fail(HYDRO_ERR_ARG, "smax_device: NULL argument%s%s");
    *smax = reinterpret_cast<double *>(&h->scal->smax_bits);
    return HYDRO_OK;
}

int hydro_reduce_smax(hydro_t *h)
{
    if (!h) return fail(HYDRO_ERR_ARG, "reduce_smax: NULL handle%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "reduce_smax before set_state%s%s");
    if (h->smax_valid) return HYDRO_OK;
    return launch_cfl_reduce(h);
}

// One substep of the RK2 step on the planes of `part`, for drivers that put a halo exchange between
// the substeps.  dt > 0: host-supplied step; dt == 0: the device-resident step, formed at the start
// of substep 1 from the (all-reduced) running maximum.
int hydro_substep(hydro_t *h, int stage, double dt, int part)
{
    if (!h || (stage != 1 && stage != 2) || part < 0 || part > 2 || !(dt >= 0.0) || !std::isfinite(dt))
        return fail(HYDRO_ERR_ARG, "substep: bad argument%s%s");
    if (!h->have_state) return fail(HYDRO_ERR_NOSTATE, "substep before set_state%s%s");
    const Grid &g = h->g;
    const bool dev_dt = dt == 0.0;
    int rc;
    if (dev_dt && !h->smax_valid) return fail(HYDRO_ERR_NOSTATE, "substep: device dt needs hydro_reduce_smax first%s%s");
    if (dev_dt && !h->t_on_device && (rc = begin_run(h, HUGE_VAL))) return rc;
    if (!dev_dt && h->t_on_device && (rc = read_scalars(h))) return rc;
    const double r = dt / h->dx;
    // interface planes: the z-chunks (fused kernel) or plane pairs (simple kernel) next to a
    // neighbouring slab; computed first so that their exchange overlaps the interior
    const int unit = (h->variant == 0 || g.ndim < 3) ? 2 : (h->plan.km < g.nz ? FUSED_SLAB_UNIT : h->plan.lz);
    int lo_end = 0, hi_begin = g.nz;
    if (g.bc[4] == HYDRO_BC_NEIGHBOUR) lo_end = unit < g.nz ? unit : g.nz;
    if (g.bc[5] == HYDRO_BC_NEIGHBOUR) {
        hi_begin = ((g.nz - 1) / unit) * unit;                   // start of the last chunk ...
        if (g.nz - hi_begin < 2 && hi_begin >= unit) hi_begin -= unit;   // ... which must hold two planes
    }
    if (hi_begin < lo_end) hi_begin = lo_end;
    const bool first = part != 2;                                // the launch that opens the substep
    if (stage == 1 && first && (rc = ensure_ghosts(h))) return rc;
    if (stage == 1 && first) {
        const int axes = fill_axes(h);
        if (axes) { if ((rc = launch_ghost_fill(h, h->A, true, dev_dt, axes))) return rc; }
        else if ((rc = launch_begin_step(h, dev_dt))) return rc;
    }
    if (stage == 2 && first) {
        const int axes = fill_axes(h);
        if (axes && (rc = launch_ghost_fill(h, h->B, false, false, axes))) return rc;
    }
    const double *in = stage == 1 ? h->A : h->B;
    const double *old = stage == 1 ? nullptr : h->A;
    double *outp = stage == 1 ? h->B : h->A;
    auto run = [&](int kb, int ke) {
        return stage == 1 ? launch_stage<1>(h, in, old, outp, r, dev_dt, false, kb, ke)
                          : launch_stage<2>(h, in, old, outp, r, dev_dt, true, kb, ke);
    };
    if (part == 0) { if ((rc = run(0, g.nz))) return rc; }
    else if (part == 1) { if ((rc = run(0, lo_end))) return rc; if ((rc = run(hi_begin, g.nz))) return rc; }
    else { if ((rc = run(lo_end, hi_begin))) return rc; }
    if (stage == 2 && (part == 0 || part == 2)) {                // the step is complete
        h->smax_valid = true;
        if (!dev_dt) { h->t = h->t + dt; h->step += 1; }
    }
    return HYDRO_OK;
}

int hydro_get_time(hydro_t *h, double *t, long long *step)
{
    if (!h) return fail(HYDRO_ERR_ARG, "get_time: NULL handle%s%s");
    int rc;
    if (h->t_on_device && (rc = read_scalars(h))) return rc;
    if (t) *t = h->t;
    if (step) *step = h->step;
    return HYDRO_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// Allocation-free entry point: hydro_max_signal_speed_noalloc (include/hydro.h).
// The CFL reduction (A8) of a packed device state for callers that cannot call cudaMalloc (CUDA graph
// capture, tight serving loops, harnesses that forbid it).  No handle, no cudaMalloc / cudaFree, no
// allocating library routine: the scratch of the reduction -- one partial maximum per block and the
// ticket that finds the last block -- lives in a file-scope device array of fixed size, which every
// GPU that loads this library holds until the process exits.
//
// In host code `g_noalloc_scratch` is a host-side stand-in for the device array, not a device address:
// the host asks cudaGetSymbolAddress for the address once per device, with that device current, and
// passes it to the kernel.  Every call on a device shares the array, which keeps the last call's
// contents: the ticket is cleared at the start of each call, partials beyond the launch's own blocks
// are never read.  Calls that overlap on the GPU (two streams, two threads) race on it.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int NOALLOC_THREADS = 256;
constexpr int NOALLOC_CELLS_PER_THREAD = 8;
constexpr long long NOALLOC_CELLS_PER_BLOCK = (long long)NOALLOC_THREADS * NOALLOC_CELLS_PER_THREAD;   // 2048
constexpr long long NOALLOC_MAX_BLOCKS = HYDRO_NOALLOC_MAX_CELLS / NOALLOC_CELLS_PER_BLOCK;            // 65536
constexpr size_t NOALLOC_HEADER_BYTES = 256;      // ticket (4 bytes used); the partials start 256-byte aligned

struct NoallocPartial { double smax; int bad; int pad; };                                               // 16 bytes

constexpr size_t NOALLOC_SCRATCH_BYTES = NOALLOC_HEADER_BYTES + (size_t)NOALLOC_MAX_BLOCKS * sizeof(NoallocPartial);
static_assert(NOALLOC_SCRATCH_BYTES == HYDRO_NOALLOC_SCRATCH_BYTES, "hydro.h states the size of the scratch array");
static_assert(NOALLOC_MAX_BLOCKS * NOALLOC_CELLS_PER_BLOCK == HYDRO_NOALLOC_MAX_CELLS, "whole blocks");

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

// One block = one chunk of 2048 cells of the packed state U[5][ncells] (coalesced: consecutive threads,
// consecutive cells); the block's maximum and unphysical flag go to partial[blockIdx.x]; the block that
// draws the last ticket folds the partials of this launch in a fixed order and writes the two outputs.
// The maximum does not depend on the order, so the result is deterministic and equal to the atomicMax
// form of cfl_reduce_kernel.
__global__ void __launch_bounds__(NOALLOC_THREADS)
cfl_reduce_noalloc_kernel(const double *__restrict__ U, long long ncells, double gamma, double gm1,
                          unsigned char *scratch, double *smax_out, int *flag_out)
{
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch);
    NoallocPartial *partial = reinterpret_cast<NoallocPartial *>(scratch + NOALLOC_HEADER_BYTES);
    __shared__ double wmax[NOALLOC_THREADS / 32];
    __shared__ int wbad[NOALLOC_THREADS / 32];
    __shared__ int is_last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;

    double s = 0.0;
    int bad = 0;
    const long long first = (long long)blockIdx.x * NOALLOC_CELLS_PER_BLOCK + threadIdx.x;
#pragma unroll
    for (int q = 0; q < NOALLOC_CELLS_PER_THREAD; ++q) {
        const long long c = first + (long long)q * NOALLOC_THREADS;
        if (c < ncells) {
            const double v = cell_signal_speed(U[c], U[ncells + c], U[2 * ncells + c], U[3 * ncells + c],
                                               U[4 * ncells + c], gamma, gm1, bad);
            s = v > s ? v : s;                 // NaN never wins; it is reported through `bad`
        }
    }
    auto fold = [&]() {                        // block-wide maximum / or into thread 0
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double other = __shfl_xor_sync(0xffffffffu, s, o);
            s = other > s ? other : s;
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (lane == 0) { wmax[wid] = s; wbad[wid] = bad; }
        __syncthreads();
        if (wid == 0) {
            s = lane < NOALLOC_THREADS / 32 ? wmax[lane] : 0.0;
            bad = lane < NOALLOC_THREADS / 32 ? wbad[lane] : 0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double other = __shfl_xor_sync(0xffffffffu, s, o);
                s = other > s ? other : s;
                bad |= __shfl_xor_sync(0xffffffffu, bad, o);
            }
        }
    };
    fold();
    if (threadIdx.x == 0) {
        partial[blockIdx.x].smax = s;
        partial[blockIdx.x].bad = bad;
        __threadfence();                       // the partial is visible before the ticket is drawn
        is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    s = 0.0;
    bad = 0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += NOALLOC_THREADS) {
        const double v = __ldcg(&partial[b].smax);
        bad |= __ldcg(&partial[b].bad);
        s = v > s ? v : s;
    }
    __syncthreads();                           // wmax / wbad are reused
    fold();
    if (threadIdx.x == 0) {
        *smax_out = s;
        *flag_out = bad ? 1 : 0;
        *ticket = 0u;                          // left clean for the next call (which clears it again)
    }
}

// Device address of the scratch array, looked up once per device (set-up) with that device current.
constexpr int NOALLOC_MAX_DEVICES = 64;
std::atomic<unsigned char *> g_noalloc_ptr[NOALLOC_MAX_DEVICES];

int noalloc_scratch(unsigned char **out)
{
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES)
        return fail(HYDRO_ERR_CUDA, "max_signal_speed_noalloc: device ordinal beyond 63%s%s");
    unsigned char *p = g_noalloc_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        // `dev` is current: the address returned is that of this device's copy of the array
        CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_noalloc_scratch));
        if (!p) return fail(HYDRO_ERR_CUDA, "max_signal_speed_noalloc: cudaGetSymbolAddress returned NULL%s%s");
        g_noalloc_ptr[dev].store(p, std::memory_order_release);   // two threads racing store the same address
    }
    *out = p;
    return HYDRO_OK;
}

// HYDRO_ERR_ARG unless `p` is memory the current device can dereference as its own (device or managed)
int noalloc_device_pointer(const void *p, const char *what)
{
    cudaPointerAttributes at;
    const cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(HYDRO_ERR_CUDA, "max_signal_speed_noalloc: cudaPointerGetAttributes(%s): %s", what, cudaGetErrorString(e));
    }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return fail(HYDRO_ERR_ARG, "max_signal_speed_noalloc: %s is not a device pointer%s", what);
    return HYDRO_OK;
}

}  // namespace

extern "C" int hydro_max_signal_speed_noalloc(const double *U_dev, long long ncells, double gamma,
                                              double *smax_dev, int *flag_dev, void *cuda_stream)
{
    // argument checks first: none of them needs a device
    if (!U_dev || !smax_dev || !flag_dev) return fail(HYDRO_ERR_ARG, "max_signal_speed_noalloc: NULL pointer%s%s");
    if (ncells < 1) return fail(HYDRO_ERR_ARG, "max_signal_speed_noalloc: ncells must be at least 1%s%s");
    if (ncells > HYDRO_NOALLOC_MAX_CELLS)
        return fail(HYDRO_ERR_ARG, "max_signal_speed_noalloc: ncells exceeds HYDRO_NOALLOC_MAX_CELLS = 134217728 (512^3), "
                                   "the capacity of the static scratch array; use a handle (hydro_max_signal_speed)%s%s");
    if (!(gamma > 1.0) || !std::isfinite(gamma)) return fail(HYDRO_ERR_ARG, "max_signal_speed_noalloc: gamma must be > 1%s%s");
    int rc;
    if ((rc = noalloc_device_pointer(U_dev, "U_dev"))) return rc;
    if ((rc = noalloc_device_pointer(smax_dev, "smax_dev"))) return rc;
    if ((rc = noalloc_device_pointer(flag_dev, "flag_dev"))) return rc;
    unsigned char *scratch = nullptr;
    if ((rc = noalloc_scratch(&scratch))) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // what must start at zero: the ticket (the header); a memset node under capture, allocates nothing
    CUDA_TRY(cudaMemsetAsync(scratch, 0, NOALLOC_HEADER_BYTES, stream));
    const unsigned blocks = (unsigned)((ncells + NOALLOC_CELLS_PER_BLOCK - 1) / NOALLOC_CELLS_PER_BLOCK);
    cfl_reduce_noalloc_kernel<<<blocks, NOALLOC_THREADS, 0, stream>>>(U_dev, ncells, gamma, gamma - 1.0, scratch,
                                                                     smax_dev, flag_dev);
    LAUNCH_CHECK("cfl_reduce_noalloc");
    return HYDRO_OK;
}
