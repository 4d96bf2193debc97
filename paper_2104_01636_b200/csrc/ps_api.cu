// ps_api.cu -- the C ABI of include/ps_poisson.h: context, workspace, launch logic.
// Every step of the path runs in the CUDA kernels of ps_kernels_*.cuh; this file only validates
// arguments, carves the workspace and enqueues launches.  There is no CPU fallback.
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/ps_poisson.h"
#include "ps_kernels_generic.cuh"
#include "ps_kernels_zmarch.cuh"
#include "ps_kernels_mg.cuh"
#include "ps_kernels_resident.cuh"
#include "ps_kernels_cluster.cuh"
#include "ps_kernels_projection.cuh"

namespace {

thread_local char g_cuda_msg[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e)
{
    snprintf(g_cuda_msg, sizeof g_cuda_msg, "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    return PS_ECUDA;
}

#define PS_CUDA(call)                                   \
    do {                                                \
        cudaError_t e_ = (call);                        \
        if (e_ != cudaSuccess) return cuda_fail(e_);    \
    } while (0)

constexpr size_t ps_resident_max_cells = 131072;

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// all pointers 16-byte aligned (the pair kernels use 16-byte loads and stores)
bool aligned16(const void *a, const void *b = nullptr, const void *c = nullptr,
               const void *d = nullptr)
{
    return (((uintptr_t)a | (uintptr_t)b | (uintptr_t)c | (uintptr_t)d) & 15u) == 0;
}

}  // namespace

struct ps_ctx {
    ps::Grid g;
    double dx, dy, dz;
    cudaStream_t stream;
    int K;                 // residual check cadence
    int variant_req;       // what the caller asked for (PS_KERNEL_*)
    int variant;           // resolved
    bool have_coef;
    bool have_rho;         // rho field of the on-the-fly sweep variant is current
    int sm_count;
    int coop;              // device supports cooperative launches
    int cluster_c;         // CTAs of the cluster kernel for this grid (0: does not fit / no device support)
    int pdl_mode;          // dependent launches of the fused sweeps: -1 automatic, 0 off, 1 on
    int pace_mode;         // pacing window of the fused sweeps: -1 automatic, 0 off, n
    long long launches;
    // workspace
    void *ws;
    size_t ws_bytes;
    bool ws_owned;
    double *ax, *ay, *az, *p_alt, *rho, *partR2, *partB2, *scal;   // scal: 3 doubles out
    unsigned *ctr;         // arrival counter of the resident kernel's grid barrier
    int nparts;
    int device;            // CUDA device the context (and every level below it) lives on
    double *h_scal;        // pinned, 4 doubles
    // staging of ps_solve_host: 3 fields, caller-owned (ps_set_host_staging) or cudaMalloc
    double *st_F, *st_rhs, *st_p;
    bool st_owned;
    // ps_solve_host: second stream for the uploads of rhs and p, which then run beside the
    // coefficient build; created on first use
    cudaStream_t copy_stream;
    cudaEvent_t copy_fork, copy_join;
    ps::ZmPlan fused;
    // optional event timing of the sweep launches (ps_enable_timing)
    bool timing;
    std::vector<cudaEvent_t> *ev;      // pairs: start, stop
    size_t ev_used;
    long long timed_launches, timed_sweeps;
    // multigrid: the next coarser level is a context of its own; lv_rhs / lv_p are the right-hand
    // side and the correction of THIS level when it is a coarse one.  Level memory (workspace of
    // every coarse context + lv_rhs + lv_p) is carved from the caller's ps_mg_set_workspace block
    // (mg_ws) or, without one, from one cudaMalloc owned by the finest context (mg_ws_owned).
    ps_ctx *child;
    double *lv_rhs, *lv_p;
    void *mg_ws;
    size_t mg_ws_bytes;
    bool mg_ws_owned;
    ps_mg_params mgp;
    int mg_nlev;           // levels in use below and including this one (0: no hierarchy)
    bool mg_ready;         // hierarchy matches the current coefficients
};

namespace {

size_t field_bytes_for(size_t cells) { return align_up(cells * sizeof(double), 256); }
size_t field_bytes(const ps_ctx *c) { return field_bytes_for(c->g.cells()); }
int nparts_for(size_t cells) { return (int)((cells + ps::RED_CHUNK - 1) / ps::RED_CHUNK); }

size_t workspace_bytes_for(size_t cells)
{
    return 5 * field_bytes_for(cells) +
           2 * align_up((size_t)nparts_for(cells) * sizeof(double), 256) + 256 + 256;
}
size_t workspace_bytes(const ps_ctx *c) { return workspace_bytes_for(c->g.cells()); }

void carve(ps_ctx *c, void *base)
{
    char *q = (char *)base;
    const size_t fb = field_bytes(c), pb = align_up((size_t)c->nparts * sizeof(double), 256);
    c->ax = (double *)q; q += fb;
    c->ay = (double *)q; q += fb;
    c->az = (double *)q; q += fb;
    c->p_alt = (double *)q; q += fb;
    c->rho = (double *)q; q += fb;
    c->partR2 = (double *)q; q += pb;
    c->partB2 = (double *)q; q += pb;
    c->scal = (double *)q; q += 256;
    c->ctr = (unsigned *)q;
}

int ensure_workspace(ps_ctx *c)
{
    if (c->ws) return PS_OK;
    void *w = nullptr;
    cudaError_t e = cudaMalloc(&w, workspace_bytes(c));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return PS_ENOMEM; }
    if (e != cudaSuccess) return cuda_fail(e);
    c->ws = w;
    c->ws_bytes = workspace_bytes(c);
    c->ws_owned = true;
    carve(c, w);
    return PS_OK;
}

// Launch options of the fused sweep when the caller leaves them to the library (measured on one
// B200 in sustained, power-capped runs of bench.py and in cold bursts; DESIGN.md 7.1,
// profiles/r02_launch_options.md):
//  * dependent launches pay where a launch is short (config 2, 8 steps per CTA: 10.2 -> 6.9 us per
//    sweep; config 3, 35 steps: 37.0 -> 35.3) and cost 4 % in sustained runs of long launches
//    (config 4, 270 steps: 129.1 -> 124.0 Gcell-updates/s at the power cap);
//  * pacing cuts the DRAM traffic of cold bursts at full clocks (config 5: 1.19 -> 1.03 x
//    algorithmic, 108 -> 134 Gcell-updates/s; config 4: 130 -> 136) and, with the counter updated
//    once per four stages, is neutral in sustained runs of long launches (config 4: 130.6 ->
//    131.1, config 5: 131.3 -> 132.8); on short launches it costs 1-2 % (config 3) to 10 %
//    (config 2).
// So: short launches (up to ps_pdl_max_steps z steps per CTA) get dependent launches, long ones
// get pacing.
constexpr int ps_pdl_max_steps = 96;

bool launch_dependent(const ps_ctx *c)
{
    return c->pdl_mode < 0 ? c->fused.pace_steps <= ps_pdl_max_steps : c->pdl_mode != 0;
}

int launch_pace_window(const ps_ctx *c)
{
    if (c->pace_mode >= 0) return c->pace_mode;
    return c->fused.pace_steps > ps_pdl_max_steps ? ps::ZM_PACE_WINDOW : 0;
}

int resolve_variant(const ps_ctx *c, int req)
{
    const bool fused_ok = c->fused.ok;
    // small grids live in L2 and are bound by launch / pipeline start-up latency: many sweeps per
    // cooperative launch win there (measured cross-over between 65 k and 524 k cells)
    if (req == PS_KERNEL_AUTO && c->cluster_c > 0) return PS_KERNEL_CLUSTER;
    if (req == PS_KERNEL_AUTO && c->coop && c->g.cells() <= (size_t)ps_resident_max_cells)
        return PS_KERNEL_RESIDENT;
    if (req == PS_KERNEL_AUTO) return fused_ok ? PS_KERNEL_FUSED : PS_KERNEL_TWOPASS;
    if (req == PS_KERNEL_FUSED && !fused_ok) return -1;
    if (req == PS_KERNEL_FUSED_OTF && !fused_ok) return -1;
    if (req == PS_KERNEL_RESIDENT && !c->coop) return -1;
    if (req == PS_KERNEL_CLUSTER && c->cluster_c == 0) return -1;
    if (req < PS_KERNEL_AUTO || req > PS_KERNEL_CLUSTER) return -1;
    return req;
}

int grid_for(const ps_ctx *c, size_t work_items, int threads)
{
    // enough blocks to cover the work once, capped at 32 resident waves of the device
    size_t blocks = (work_items + threads - 1) / threads;
    const size_t cap = (size_t)c->sm_count * 8 * 32;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    return (int)blocks;
}

// Launch geometry of the z-marching pair stencils (ps_kernels_projection.cuh): tiles of 64 cells x
// 8 rows, z chunks of *kz planes (two halo planes of one field per chunk), about `waves` blocks
// per SM in the launch.  Measured on config 4: ps_rhs_from_velocity 225 / 212 / 197 us with 8 /
// 16 / 32 blocks per SM, ps_face_divergence 376 / 388 / 382 us.
dim3 zs_grid(const ps_ctx *c, int waves, int *kz)
{
    const int tx = (c->g.nx / 2 + ps::ZS_TX - 1) / ps::ZS_TX, ty = (c->g.ny + ps::ZS_TY - 1) / ps::ZS_TY;
    const long long want = (long long)c->sm_count * waves;
    long long zc = (want + (long long)tx * ty - 1) / ((long long)tx * ty);
    const int zc_max = c->g.nz / 4 > 0 ? c->g.nz / 4 : 1;
    if (zc > zc_max) zc = zc_max;
    if (zc < 1) zc = 1;
    *kz = (c->g.nz + (int)zc - 1) / (int)zc;
    return dim3((unsigned)tx, (unsigned)ty, (unsigned)((c->g.nz + *kz - 1) / *kz));
}

int launch_half_sweep(ps_ctx *c, const double *rhs, double *p, double omega, int colour)
{
    const size_t items = (size_t)((c->g.nx + 1) / 2) * c->g.ny * c->g.nz;
    ps::ps_half_sweep_kernel<<<grid_for(c, items, 256), 256, 0, c->stream>>>(
        c->g, c->ax, c->ay, c->az, rhs, p, omega, colour);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

// n sweeps, any variant.  The in-place variants work on *cur.  The fused variants ping-pong
// between the caller's p and p_alt: *cur is the buffer that holds the iterate on entry and on
// return (p or c->p_alt); callers copy back to p once, when they are done (settle_p).
int run_sweeps_untimed(ps_ctx *c, const double *rhs, double *p, double **cur, double omega, int n);

int run_sweeps(ps_ctx *c, const double *rhs, double *p, double **cur, double omega, int n)
{
    if (n <= 0) return PS_OK;
    if (!c->timing) return run_sweeps_untimed(c, rhs, p, cur, omega, n);
    if (c->ev_used + 2 > c->ev->size()) {
        cudaEvent_t a, b;
        PS_CUDA(cudaEventCreate(&a));
        PS_CUDA(cudaEventCreate(&b));
        c->ev->push_back(a);
        c->ev->push_back(b);
    }
    const long long before = c->launches;
    PS_CUDA(cudaEventRecord((*c->ev)[c->ev_used], c->stream));
    const int rc = run_sweeps_untimed(c, rhs, p, cur, omega, n);
    PS_CUDA(cudaEventRecord((*c->ev)[c->ev_used + 1], c->stream));
    c->ev_used += 2;
    c->timed_launches += c->launches - before;
    c->timed_sweeps += n;
    return rc;
}

int run_sweeps_untimed(ps_ctx *c, const double *rhs, double *p, double **cur, double omega, int n)
{
    if (c->variant == PS_KERNEL_TWOPASS) {
        for (int s = 0; s < n; ++s) {
            int rc = launch_half_sweep(c, rhs, *cur, omega, 0);
            if (rc) return rc;
            rc = launch_half_sweep(c, rhs, *cur, omega, 1);
            if (rc) return rc;
        }
        return PS_OK;
    }
    if (c->variant == PS_KERNEL_CLUSTER) {
        const cudaError_t e = ps::cl_launch(c->g, c->cluster_c, c->ax, c->ay, c->az, rhs, *cur,
                                            omega, n, c->stream);
        c->launches++;
        return e == cudaSuccess ? PS_OK : cuda_fail(e);
    }
    if (c->variant == PS_KERNEL_RESIDENT) {
        const size_t items = (size_t)((c->g.nx + 1) / 2) * c->g.ny * c->g.nz;
        int threads = ps::RES_THREADS;
        size_t blocks = (items + threads - 1) / threads;
        if (items <= (size_t)ps::RES_THREADS_ONE) { threads = ps::RES_THREADS_ONE; blocks = 1; }
        if (blocks > (size_t)c->sm_count) blocks = (size_t)c->sm_count;
        if ((long long)n * 2 * (long long)blocks > 0x7fffffffLL) return PS_EINVAL;
        ps::Grid g = c->g;
        const double *ax = c->ax, *ay = c->ay, *az = c->az;
        double *pp = *cur;
        unsigned *ctr = c->ctr;
        if (blocks > 1) PS_CUDA(cudaMemsetAsync(ctr, 0, sizeof(unsigned), c->stream));
        void *args[] = {&g, &ax, &ay, &az, &rhs, &pp, &omega, &n, &ctr};
        PS_CUDA(cudaLaunchCooperativeKernel((const void *)ps::ps_resident_sweeps_kernel,
                                            dim3((unsigned)blocks), dim3((unsigned)threads), args,
                                            0, c->stream));
        c->launches++;
        return PS_OK;
    }
    double *src = *cur, *dst = (src == p) ? c->p_alt : p;
    const bool otf = c->variant == PS_KERNEL_FUSED_OTF;
    if (otf && !c->have_rho) return PS_ESTATE;
    const double c2x = 2.0 * (1.0 / (c->dx * c->dx)), c2y = 2.0 * (1.0 / (c->dy * c->dy)),
                 c2z = 2.0 * (1.0 / (c->dz * c->dz));
    const bool pdl_on = launch_dependent(c);
    c->fused.pace_window = launch_pace_window(c);
    for (int left = n; left > 0; --left) {
        // every sweep after the first of the batch is a dependent launch: its predecessor in the
        // stream is a sweep, which writes none of the coefficient, rho or rhs boxes
        const bool dep = pdl_on && left < n;
        cudaError_t e =
            otf ? ps::zm_launch_otf(c->fused, c->g, c->rho, c2x, c2y, c2z, rhs, src, dst, omega,
                                    c->stream, dep)
                : ps::zm_launch(c->fused, c->g, c->ax, c->ay, c->az, rhs, src, dst, omega,
                                c->stream, dep);
        c->launches++;
        if (e != cudaSuccess) return cuda_fail(e);
        double *t = src; src = dst; dst = t;
    }
    *cur = src;
    return PS_OK;
}

// Bring the iterate back into the caller's p if the ping-pong left it in p_alt.
int settle_p(ps_ctx *c, double *p, double **cur)
{
    if (*cur != p) {
        PS_CUDA(cudaMemcpyAsync(p, *cur, c->g.cells() * sizeof(double), cudaMemcpyDeviceToDevice,
                                c->stream));
        *cur = p;
    }
    return PS_OK;
}

// n sweeps in place on the caller's p (one device copy at the end if the ping-pong count is odd)
int run_sweeps_inplace(ps_ctx *c, const double *rhs, double *p, double omega, int n)
{
    double *cur = p;
    const int rc = run_sweeps(c, rhs, p, &cur, omega, n);
    return rc ? rc : settle_p(c, p, &cur);
}

int enqueue_residual(ps_ctx *c, const double *rhs, const double *p)
{
    // the summation tree is a function of the grid shape alone (every *_dev pointer is 16-byte
    // aligned: checked at the ABI), so the norm of given data never depends on where it lives
    if (c->g.nx % 2 == 0)
        ps::ps_residual_partial_pair_kernel<<<c->nparts, ps::RED_THREADS, 0, c->stream>>>(
            c->g, c->ax, c->ay, c->az, rhs, p, c->partR2, c->partB2);
    else
        ps::ps_residual_partial_kernel<<<c->nparts, ps::RED_THREADS, 0, c->stream>>>(
            c->g, c->ax, c->ay, c->az, rhs, p, c->partR2, c->partB2);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    ps::ps_reduce_final_kernel<<<1, ps::FIN_THREADS, 0, c->stream>>>(c->partR2, c->partB2,
                                                                    c->nparts, c->scal);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    PS_CUDA(cudaMemcpyAsync(c->h_scal, c->scal, 3 * sizeof(double), cudaMemcpyDeviceToHost,
                            c->stream));
    return PS_OK;
}

}  // namespace

extern "C" {

int ps_create(ps_ctx **out, int nx, int ny, int nz, double dx, double dy, double dz)
{
    if (!out) return PS_EINVAL;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 2 || (nz & 1)) return PS_EINVAL;
    if (!(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0) || !std::isfinite(dx) || !std::isfinite(dy) ||
        !std::isfinite(dz))
        return PS_EINVAL;
    if ((double)nx * (double)ny * (double)nz > 2.0e9) return PS_EINVAL;
    int dev = 0, sms = 0;
    PS_CUDA(cudaGetDevice(&dev));
    PS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    int coop = 0;
    PS_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    ps_ctx *c = new (std::nothrow) ps_ctx();
    if (!c) return PS_ENOMEM;
    c->g = ps::Grid{nx, ny, nz};
    c->device = dev;
    c->ev = new (std::nothrow) std::vector<cudaEvent_t>();
    if (!c->ev) { delete c; return PS_ENOMEM; }
    c->dx = dx; c->dy = dy; c->dz = dz;
    c->K = 50;
    c->pdl_mode = -1;
    c->pace_mode = -1;
    c->sm_count = sms;
    c->coop = coop;
    c->nparts = nparts_for(c->g.cells());
    cudaError_t e = cudaMallocHost((void **)&c->h_scal, 4 * sizeof(double));
    if (e != cudaSuccess) { delete c->ev; delete c; return cuda_fail(e); }
    e = ps::zm_plan_init(&c->fused, c->g, sms);
    if (e != cudaSuccess) {
        ps::zm_plan_destroy(&c->fused);
        cudaFreeHost(c->h_scal);
        delete c->ev;
        delete c;
        return cuda_fail(e);
    }
    c->cluster_c = ps::cl_plan(c->g);
    c->variant_req = PS_KERNEL_AUTO;
    c->variant = resolve_variant(c, PS_KERNEL_AUTO);
    *out = c;
    return PS_OK;
}

int ps_destroy(ps_ctx *c)
{
    if (!c) return PS_OK;
    if (c->child) ps_destroy(c->child);
    if (c->mg_ws && c->mg_ws_owned) cudaFree(c->mg_ws);
    if (c->ws && c->ws_owned) cudaFree(c->ws);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    ps::zm_plan_destroy(&c->fused);
    if (c->st_F && c->st_owned) cudaFree(c->st_F);
    if (c->copy_stream) {
        cudaStreamDestroy(c->copy_stream);
        cudaEventDestroy(c->copy_fork);
        cudaEventDestroy(c->copy_join);
    }
    if (c->ev) {
        for (cudaEvent_t e : *c->ev) cudaEventDestroy(e);
        delete c->ev;
    }
    delete c;
    return PS_OK;
}

size_t ps_workspace_bytes(const ps_ctx *c) { return c ? workspace_bytes(c) : 0; }

int ps_set_workspace(ps_ctx *c, void *ws_dev, size_t bytes)
{
    if (!c || !ws_dev) return PS_EINVAL;
    if (((uintptr_t)ws_dev & 255u) != 0 || bytes < workspace_bytes(c)) return PS_EINVAL;
    if (c->ws && c->ws_owned) cudaFree(c->ws);
    c->ws = ws_dev;
    c->ws_bytes = bytes;
    c->ws_owned = false;
    c->have_coef = false;
    c->have_rho = false;
    c->mg_ready = false;
    carve(c, ws_dev);
    return PS_OK;
}

int ps_set_stream(ps_ctx *c, void *cuda_stream)
{
    if (!c) return PS_EINVAL;
    c->stream = (cudaStream_t)cuda_stream;
    return PS_OK;
}

int ps_set_check_interval(ps_ctx *c, int K)
{
    if (!c || K < 1) return PS_EINVAL;
    c->K = K;
    return PS_OK;
}

int ps_set_kernel(ps_ctx *c, int variant)
{
    if (!c) return PS_EINVAL;
    const int v = resolve_variant(c, variant);
    if (v < 0) return PS_EINVAL;
    c->variant_req = variant;
    c->variant = v;
    return PS_OK;
}

int ps_get_kernel(const ps_ctx *c) { return c ? c->variant : PS_EINVAL; }

int ps_set_tuning(ps_ctx *c, int rows_per_thread, int z_chunks)
{
    if (!c || !c->fused.ok) return PS_EINVAL;
    if (rows_per_thread < 0 || rows_per_thread > 1 || z_chunks < 0 || z_chunks > c->g.nz / 2)
        return PS_EINVAL;
    PS_CUDA(cudaStreamSynchronize(c->stream));
    const cudaError_t e = ps::zm_plan_tiles(&c->fused, c->g, z_chunks);
    if (e == cudaErrorInvalidValue) { cudaGetLastError(); return PS_EINVAL; }
    if (e != cudaSuccess) return cuda_fail(e);
    return PS_OK;
}

int ps_get_tuning(const ps_ctx *c, int *rows_per_thread, int *z_chunks, int *tiles, int *ctas,
                  int *items)
{
    if (!c || !c->fused.ok) return PS_EINVAL;
    if (rows_per_thread) *rows_per_thread = 1;
    if (z_chunks) *z_chunks = c->fused.forced ? c->fused.nchunks : 0;
    if (tiles) *tiles = c->fused.ntiles;
    if (ctas) *ctas = c->fused.ncta;
    if (items) *items = c->fused.nitems;
    return PS_OK;
}

int ps_set_launch_options(ps_ctx *c, int dependent_launch, int pace_window)
{
    if (!c || !c->fused.ok) return PS_EINVAL;
    if (dependent_launch < -1 || dependent_launch > 1 || pace_window < -1 || pace_window > 64)
        return PS_EINVAL;
    c->pdl_mode = dependent_launch;
    c->pace_mode = pace_window;
    // forget an earlier "a CTA gave up waiting" (zm_pace): the caller asks for pacing afresh
    if (c->fused.d_pace)
        PS_CUDA(cudaMemsetAsync(c->fused.d_pace + 1, 0, sizeof(unsigned long long), c->stream));
    return PS_OK;
}

int ps_get_launch_options(const ps_ctx *c, int *dependent_launch, int *pace_window)
{
    if (!c || !c->fused.ok) return PS_EINVAL;
    if (dependent_launch) *dependent_launch = launch_dependent(c) ? 1 : 0;
    if (pace_window) *pace_window = launch_pace_window(c);
    return PS_OK;
}

int ps_fused_plan(int nx, int ny, int nz, int sm_count, int z_chunks, int *tiles_out, int tile_cap,
                  int *items_out, int item_cap, int *ntiles, int *nitems, int *nctas)
{
    if (nx < 1 || ny < 1 || nz < 2 || (nz & 1) || sm_count < 1 || z_chunks < 0 || !ntiles ||
        !nitems || !nctas)
        return PS_EINVAL;
    const ps::Grid g{nx, ny, nz};
    if (!ps::zm_shape_ok(g)) return PS_EINVAL;
    std::vector<ps::ZmTile> tiles;
    std::vector<ps::ZmItem> items;
    std::vector<int> first;
    int tx = 0, ty = 0, nch = 0, rec = 0;
    if (!ps::zm_plan_host(g, sm_count, z_chunks, tiles, items, first, &tx, &ty, &nch, &rec))
        return PS_EINVAL;
    *ntiles = (int)tiles.size();
    *nitems = (int)items.size();
    *nctas = (int)first.size() - 1;
    if (tiles_out)
        for (int q = 0; q < *ntiles && q < tile_cap; ++q) {
            tiles_out[4 * q] = tiles[q].xs; tiles_out[4 * q + 1] = tiles[q].xe;
            tiles_out[4 * q + 2] = tiles[q].ys; tiles_out[4 * q + 3] = tiles[q].ye;
        }
    if (items_out)
        for (int b = 0; b + 1 < (int)first.size(); ++b)
            for (int q = first[b]; q < first[b + 1] && q < item_cap; ++q) {
                items_out[4 * q] = b; items_out[4 * q + 1] = items[q].tile;
                items_out[4 * q + 2] = items[q].ks; items_out[4 * q + 3] = items[q].ke;
            }
    return PS_OK;
}

int ps_set_fraction(ps_ctx *c, const double *F_dev, double rho_l, double rho_g)
{
    if (!c || !F_dev || !aligned16(F_dev)) return PS_EINVAL;
    if (!(rho_l > 0.0) || !(rho_g > 0.0) || !std::isfinite(rho_l) || !std::isfinite(rho_g))
        return PS_EINVAL;
    int rc = ensure_workspace(c);
    if (rc) return rc;
    const double cx = 1.0 / (c->dx * c->dx), cy = 1.0 / (c->dy * c->dy), cz = 1.0 / (c->dz * c->dz);
    if (c->g.nx % 2 == 0)
        ps::ps_coef_build_pair_kernel<<<grid_for(c, c->g.cells() / 2, 256), 256, 0, c->stream>>>(
            c->g, cx, cy, cz, rho_l, rho_g, F_dev, c->ax, c->ay, c->az);
    else
        ps::ps_coef_build_kernel<<<grid_for(c, c->g.cells(), 256), 256, 0, c->stream>>>(
            c->g, cx, cy, cz, rho_l, rho_g, F_dev, c->ax, c->ay, c->az);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    c->have_rho = false;
    if (c->variant == PS_KERNEL_FUSED_OTF) {
        ps::ps_rho_build_kernel<<<grid_for(c, c->g.cells(), 256), 256, 0, c->stream>>>(
            c->g.cells(), rho_l, rho_g, F_dev, c->rho);
        c->launches++;
        PS_CUDA(cudaGetLastError());
        c->have_rho = true;
    }
    c->have_coef = true;
    c->mg_ready = false;
    return PS_OK;
}

int ps_export_coefficients(ps_ctx *c, double *ax_dev, double *ay_dev, double *az_dev)
{
    if (!c) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    const size_t b = c->g.cells() * sizeof(double);
    if (ax_dev) PS_CUDA(cudaMemcpyAsync(ax_dev, c->ax, b, cudaMemcpyDeviceToDevice, c->stream));
    if (ay_dev) PS_CUDA(cudaMemcpyAsync(ay_dev, c->ay, b, cudaMemcpyDeviceToDevice, c->stream));
    if (az_dev) PS_CUDA(cudaMemcpyAsync(az_dev, c->az, b, cudaMemcpyDeviceToDevice, c->stream));
    return PS_OK;
}

int ps_sweeps(ps_ctx *c, const double *rhs_dev, double *p_dev, double omega, int n)
{
    if (!c || !rhs_dev || !p_dev || n < 0 || !aligned16(rhs_dev, p_dev)) return PS_EINVAL;
    if (!(omega > 0.0 && omega < 2.0)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    return run_sweeps_inplace(c, rhs_dev, p_dev, omega, n);
}

int ps_half_sweep(ps_ctx *c, const double *rhs_dev, double *p_dev, double omega, int colour)
{
    if (!c || !rhs_dev || !p_dev || (colour != 0 && colour != 1)) return PS_EINVAL;
    if (!aligned16(rhs_dev, p_dev) || !(omega > 0.0 && omega < 2.0)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    return launch_half_sweep(c, rhs_dev, p_dev, omega, colour);
}

int ps_residual(ps_ctx *c, const double *rhs_dev, const double *p_dev, double *res_abs,
                double *res_rel, double *rhs_norm)
{
    if (!c || !rhs_dev || !p_dev || !res_abs || !aligned16(rhs_dev, p_dev)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    int rc = enqueue_residual(c, rhs_dev, p_dev);
    if (rc) return rc;
    PS_CUDA(cudaStreamSynchronize(c->stream));
    *res_abs = c->h_scal[0];
    if (res_rel) *res_rel = c->h_scal[1];
    if (rhs_norm) *rhs_norm = c->h_scal[2];
    return PS_OK;
}

int ps_solve(ps_ctx *c, const double *rhs_dev, double *p_dev, double omega, int max_sweeps,
             double tol, ps_info *info)
{
    if (!c || !rhs_dev || !p_dev || max_sweeps < 0 || !aligned16(rhs_dev, p_dev)) return PS_EINVAL;
    if (!(omega > 0.0 && omega < 2.0)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    int s = 0, converged = 0, rc = 0;
    bool checked = false;
    // the fused kernels ping-pong between p_dev and p_alt; the checks read whichever buffer holds
    // the iterate, and p_dev is brought up to date once, at the end (no copy per odd batch)
    double *cur = p_dev;
    if (tol > 0.0) {
        while (s < max_sweeps) {
            const int batch = (max_sweeps - s < c->K) ? (max_sweeps - s) : c->K;   // next check
            rc = run_sweeps(c, rhs_dev, p_dev, &cur, omega, batch);
            if (rc) return rc;
            s += batch;
            rc = enqueue_residual(c, rhs_dev, cur);
            if (rc) return rc;
            PS_CUDA(cudaStreamSynchronize(c->stream));
            checked = true;
            if (c->h_scal[1] <= tol) { converged = 1; break; }
        }
    } else {
        rc = run_sweeps(c, rhs_dev, p_dev, &cur, omega, max_sweeps);
        if (rc) return rc;
        s = max_sweeps;
    }
    if ((rc = settle_p(c, p_dev, &cur))) return rc;
    if (!checked) {
        rc = enqueue_residual(c, rhs_dev, p_dev);
        if (rc) return rc;
        if (tol > 0.0) {
            PS_CUDA(cudaStreamSynchronize(c->stream));
            if (c->h_scal[1] <= tol) converged = 1;
        }
    }
    PS_CUDA(cudaStreamSynchronize(c->stream));
    if (info) {
        info->sweeps = s;
        info->converged = converged;
        info->res_abs = c->h_scal[0];
        info->res_rel = c->h_scal[1];
        info->rhs_norm = c->h_scal[2];
    }
    return PS_OK;
}

size_t ps_host_staging_bytes(const ps_ctx *c) { return c ? 3 * field_bytes(c) : 0; }

int ps_set_host_staging(ps_ctx *c, void *st_dev, size_t bytes)
{
    if (!c || !st_dev) return PS_EINVAL;
    if (((uintptr_t)st_dev & 255u) != 0 || bytes < 3 * field_bytes(c)) return PS_EINVAL;
    if (c->st_F && c->st_owned) cudaFree(c->st_F);
    c->st_F = (double *)st_dev;
    c->st_rhs = (double *)((char *)st_dev + field_bytes(c));
    c->st_p = (double *)((char *)st_dev + 2 * field_bytes(c));
    c->st_owned = false;
    return PS_OK;
}

int ps_solve_host(ps_ctx *c, const double *F_host, double rho_l, double rho_g,
                  const double *rhs_host, double *p_host, double omega, int max_sweeps,
                  double tol, ps_info *info)
{
    if (!c || !F_host || !rhs_host || !p_host) return PS_EINVAL;
    const size_t b = c->g.cells() * sizeof(double);
    if (!c->st_F) {
        void *st = nullptr;
        const cudaError_t e = cudaMalloc(&st, 3 * field_bytes(c));
        if (e != cudaSuccess) {
            cudaGetLastError();
            return e == cudaErrorMemoryAllocation ? PS_ENOMEM : cuda_fail(e);
        }
        ps_set_host_staging(c, st, 3 * field_bytes(c));
        c->st_owned = true;
    }
    if (!c->copy_stream) {
        PS_CUDA(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        PS_CUDA(cudaEventCreateWithFlags(&c->copy_fork, cudaEventDisableTiming));
        PS_CUDA(cudaEventCreateWithFlags(&c->copy_join, cudaEventDisableTiming));
    }
    // F first; rhs and p follow on the copy stream (ordered after F and after everything already
    // queued on the context's stream), so the coefficient build runs beside their upload
    PS_CUDA(cudaMemcpyAsync(c->st_F, F_host, b, cudaMemcpyHostToDevice, c->stream));
    PS_CUDA(cudaEventRecord(c->copy_fork, c->stream));
    PS_CUDA(cudaStreamWaitEvent(c->copy_stream, c->copy_fork, 0));
    PS_CUDA(cudaMemcpyAsync(c->st_rhs, rhs_host, b, cudaMemcpyHostToDevice, c->copy_stream));
    PS_CUDA(cudaMemcpyAsync(c->st_p, p_host, b, cudaMemcpyHostToDevice, c->copy_stream));
    PS_CUDA(cudaEventRecord(c->copy_join, c->copy_stream));
    int rc = ps_set_fraction(c, c->st_F, rho_l, rho_g);
    PS_CUDA(cudaStreamWaitEvent(c->stream, c->copy_join, 0));
    if (rc) return rc;
    rc = ps_solve(c, c->st_rhs, c->st_p, omega, max_sweeps, tol, info);
    if (rc) return rc;
    PS_CUDA(cudaMemcpyAsync(p_host, c->st_p, b, cudaMemcpyDeviceToHost, c->stream));
    PS_CUDA(cudaStreamSynchronize(c->stream));
    return PS_OK;
}

int ps_enable_timing(ps_ctx *c, int on)
{
    if (!c) return PS_EINVAL;
    c->timing = on != 0;
    return PS_OK;
}

int ps_timing(ps_ctx *c, double *sweep_ms, long long *sweep_launches, long long *sweeps)
{
    if (!c) return PS_EINVAL;
    PS_CUDA(cudaStreamSynchronize(c->stream));
    double tot = 0.0;
    for (size_t q = 0; q + 1 < c->ev_used; q += 2) {
        float ms = 0.f;
        PS_CUDA(cudaEventElapsedTime(&ms, (*c->ev)[q], (*c->ev)[q + 1]));
        tot += (double)ms;
    }
    if (sweep_ms) *sweep_ms = tot;
    if (sweep_launches) *sweep_launches = c->timed_launches;
    if (sweeps) *sweeps = c->timed_sweeps;
    c->ev_used = 0;
    c->timed_launches = 0;
    c->timed_sweeps = 0;
    return PS_OK;
}

int ps_checked_build(void)
{
#ifdef PS_CHECKED
    return 1;
#else
    return 0;
#endif
}

int ps_debug_sabotage(ps_ctx *c, int mode)
{
    if (!c || mode < 0 || mode > 2) return PS_EINVAL;
#ifdef PS_CHECKED
    c->fused.sabotage = mode;
    return PS_OK;
#else
    return mode == 0 ? PS_OK : PS_EINVAL;           // the product build has no such switch
#endif
}

int ps_debug_read(ps_ctx *c, unsigned long long *out_host)
{
    if (!c || !out_host) return PS_EINVAL;
    for (int q = 0; q < 8; ++q) out_host[q] = 0;
    if (!c->fused.d_dbg) return PS_OK;              // product build / grid without fused kernel
    PS_CUDA(cudaStreamSynchronize(c->stream));
    PS_CUDA(cudaMemcpy(out_host, c->fused.d_dbg, 8 * sizeof(unsigned long long),
                       cudaMemcpyDeviceToHost));
    for (ps_ctx *k = c->child; k; k = k->child) {   // multigrid levels: add their counts
        unsigned long long t[8] = {0};
        if (!k->fused.d_dbg) continue;
        PS_CUDA(cudaMemcpy(t, k->fused.d_dbg, sizeof t, cudaMemcpyDeviceToHost));
        if (out_host[0] == 0 && t[0] != 0)
            for (int q = 1; q < 8; ++q) out_host[q] = t[q];
        out_host[0] += t[0];
    }
    return PS_OK;
}

long long ps_launch_count(const ps_ctx *c)
{
    long long n = 0;
    for (; c; c = c->child) n += c->launches;
    return n;
}

}  // extern "C"

// ----------------------------------------------------------------------------- multigrid
namespace {

int mg_max_levels(int nx, int ny, int nz)
{
    int L = 1;
    while (nx % 2 == 0 && ny % 2 == 0 && nz % 4 == 0 && nx / 2 >= 2 && ny / 2 >= 2) {
        nx /= 2; ny /= 2; nz /= 2; ++L;
    }
    return L;
}

// device bytes of the coarse levels 1 .. nlev-1 of a hierarchy on grid g: per level the context's
// own workspace (coefficients, ping-pong buffer, partials) + its right-hand side + its correction
size_t mg_bytes(ps::Grid g, int nlev)
{
    size_t tot = 0;
    for (int l = 1; l < nlev; ++l) {
        g = ps::Grid{g.nx / 2, g.ny / 2, g.nz / 2};
        tot += workspace_bytes_for(g.cells()) + 2 * field_bytes_for(g.cells());
    }
    return tot;
}

void mg_drop_levels(ps_ctx *c)
{
    if (c->child) ps_destroy(c->child);
    c->child = nullptr;
    c->mg_nlev = 0;
    c->mg_ready = false;
}

// Create the contexts of levels 1 .. nlev-1 below c and hand each its slice of the level block
// (the caller's ps_mg_set_workspace block, else one cudaMalloc owned by c).
int mg_build_levels(ps_ctx *c, int nlev)
{
    const size_t need = mg_bytes(c->g, nlev);
    if (need > 0) {
        if (c->mg_ws && !c->mg_ws_owned && c->mg_ws_bytes < need) return PS_EINVAL;
        if (c->mg_ws && c->mg_ws_owned && c->mg_ws_bytes < need) {
            cudaFree(c->mg_ws);
            c->mg_ws = nullptr;
        }
        if (!c->mg_ws) {
            const cudaError_t e = cudaMalloc(&c->mg_ws, need);
            if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); c->mg_ws = nullptr; return PS_ENOMEM; }
            if (e != cudaSuccess) { c->mg_ws = nullptr; return cuda_fail(e); }
            c->mg_ws_bytes = need;
            c->mg_ws_owned = true;
        }
    }
    char *q = (char *)c->mg_ws;
    ps_ctx *f = c;
    for (int l = 1; l < nlev; ++l) {
        ps_ctx *k = nullptr;
        int rc = ps_create(&k, f->g.nx / 2, f->g.ny / 2, f->g.nz / 2, 2.0 * f->dx, 2.0 * f->dy,
                           2.0 * f->dz);
        if (rc) return rc;
        f->child = k;
        if ((rc = ps_set_workspace(k, q, workspace_bytes(k)))) return rc;
        q += workspace_bytes(k);
        k->lv_rhs = (double *)q; q += field_bytes(k);
        k->lv_p = (double *)q; q += field_bytes(k);
        f = k;
    }
    return PS_OK;
}

int mg_launch_coarsen(ps_ctx *f, ps_ctx *k)
{
    ps::ps_mg_coarsen_kernel<<<grid_for(f, k->g.cells(), 256), 256, 0, f->stream>>>(
        f->g, f->ax, f->ay, f->az, k->ax, k->ay, k->az);
    f->launches++;
    PS_CUDA(cudaGetLastError());
    k->have_coef = true;
    return PS_OK;
}

int mg_launch_residual_restrict(ps_ctx *f, const double *rhs, const double *p, double *rc)
{
    ps::ps_mg_residual_restrict_pair_kernel<<<grid_for(f, f->g.cells() / 8, 256), 256, 0,
                                              f->stream>>>(f->g, f->ax, f->ay, f->az, rhs, p, rc);
    f->launches++;
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

int mg_launch_prolong_add(ps_ctx *f, const double *ec, double *p)
{
    ps::ps_mg_prolong_add_kernel<<<grid_for(f, f->g.cells() / 2, 256), 256, 0, f->stream>>>(
        f->g, ec, p);
    f->launches++;
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

int mg_nu(int nu, int level, const ps_mg_params &m)
{
    const int cap = (level >= 2 && m.nu_max_deep < m.nu_max) ? m.nu_max_deep : m.nu_max;
    long long v = nu;
    for (int q = 0; q < level && v < cap; ++q) v *= m.nu_growth;
    return (int)(v < cap ? v : (nu < cap ? cap : nu));
}

// The finest level of ps_mg_solve may take its norm inside the residual + restriction pass: with
// no pre-smoothing there (nu1 = 0) the residual that is restricted is the residual of the
// iterate the stopping test looks at.
bool mg_fused_norm_ok(const ps_ctx *f)
{
    return f->child && f->mg_nlev > 1 && mg_nu(f->mgp.nu1, 0, f->mgp) == 0;
}

// residual + restriction + norm partials of level f, then the final reduction and the read-back
int mg_launch_residual_restrict_norm(ps_ctx *f, const double *rhs, const double *p, double *rc)
{
    ps::ps_mg_residual_restrict_norm_kernel<<<f->nparts, ps::RED_THREADS, 0, f->stream>>>(
        f->g, f->ax, f->ay, f->az, rhs, p, rc, f->partR2, f->partB2);
    f->launches++;
    PS_CUDA(cudaGetLastError());
    ps::ps_reduce_final_kernel<<<1, ps::FIN_THREADS, 0, f->stream>>>(f->partR2, f->partB2,
                                                                    f->nparts, f->scal);
    f->launches++;
    PS_CUDA(cudaGetLastError());
    PS_CUDA(cudaMemcpyAsync(f->h_scal, f->scal, 3 * sizeof(double), cudaMemcpyDeviceToHost,
                            f->stream));
    return PS_OK;
}

// M6: one cycle on the level of context f (level index = depth below the finest).  restricted:
// the right-hand side of the next level has already been written (fused norm path, level 0).
int mg_cycle(ps_ctx *f, const ps_mg_params &m, const double *rhs, double *p, int level = 0,
             bool restricted = false)
{
    int rc;
    const double omega = level == 0 ? m.omega_s : m.omega_c;
    if (!f->child || f->mg_nlev <= 1)
        return run_sweeps_inplace(f, rhs, p, omega, m.coarse_sweeps);
    ps_ctx *k = f->child;
    if (!restricted) {
        if ((rc = run_sweeps_inplace(f, rhs, p, omega, mg_nu(m.nu1, level, m)))) return rc;
        if ((rc = mg_launch_residual_restrict(f, rhs, p, k->lv_rhs))) return rc;
    }
    PS_CUDA(cudaMemsetAsync(k->lv_p, 0, k->g.cells() * sizeof(double), f->stream));
    for (int g = 0; g < m.gamma; ++g)
        if ((rc = mg_cycle(k, m, k->lv_rhs, k->lv_p, level + 1))) return rc;
    if ((rc = mg_launch_prolong_add(f, k->lv_p, p))) return rc;
    return run_sweeps_inplace(f, rhs, p, omega, mg_nu(m.nu2, level, m));
}

}  // namespace

extern "C" {

size_t ps_mg_workspace_bytes(const ps_ctx *c, int levels)
{
    if (!c) return 0;
    const int maxl = mg_max_levels(c->g.nx, c->g.ny, c->g.nz);
    const int nlev = levels > maxl ? maxl : (levels < 1 ? 1 : levels);
    return mg_bytes(c->g, nlev);
}

int ps_mg_set_workspace(ps_ctx *c, void *ws_dev, size_t bytes)
{
    if (!c || !ws_dev || ((uintptr_t)ws_dev & 255u) != 0) return PS_EINVAL;
    mg_drop_levels(c);                       // the old levels point into the old block
    if (c->mg_ws && c->mg_ws_owned) cudaFree(c->mg_ws);
    c->mg_ws = ws_dev;
    c->mg_ws_bytes = bytes;
    c->mg_ws_owned = false;
    return PS_OK;
}

int ps_mg_setup(ps_ctx *c, const ps_mg_params *prm)
{
    if (!c || !prm) return PS_EINVAL;
    if (prm->nu1 < 0 || prm->nu2 < 0 || prm->nu_growth < 1 || prm->nu_max < 1 ||
        prm->nu_max_deep < 1 ||
        prm->coarse_sweeps < 1 || prm->gamma < 1 ||
        prm->gamma > 2 || !(prm->omega_s > 0.0 && prm->omega_s < 2.0) ||
        !(prm->omega_c > 0.0 && prm->omega_c < 2.0) || prm->stall_cycles < 0 ||
        !(prm->omega_c_step >= 0.0) || !std::isfinite(prm->omega_c_step))
        return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    int dev = -1;
    PS_CUDA(cudaGetDevice(&dev));
    if (dev != c->device) return PS_EINVAL;    // the levels must live on the context's device
    c->mg_ready = false;
    int nlev = prm->levels;
    const int maxl = mg_max_levels(c->g.nx, c->g.ny, c->g.nz);
    if (nlev > maxl) nlev = maxl;
    if (nlev < 1) nlev = 1;
    if (c->mg_nlev != nlev) {                  // first set-up or another depth: (re)build the chain
        mg_drop_levels(c);
        const int rc = mg_build_levels(c, nlev);
        if (rc) { mg_drop_levels(c); return rc; }
    }
    ps_ctx *f = c;
    for (int l = 0; l < nlev; ++l) {
        f->mg_nlev = nlev - l;
        f->mgp = *prm;
        if (l == nlev - 1) break;
        f->child->stream = c->stream;
        const int rc = mg_launch_coarsen(f, f->child);
        if (rc) return rc;
        f = f->child;
    }
    c->mg_ready = true;
    return PS_OK;
}

int ps_mg_levels(const ps_ctx *c) { return c ? c->mg_nlev : 0; }

int ps_mg_solve(ps_ctx *c, const double *rhs_dev, double *p_dev, int max_cycles, double tol,
                ps_info *info)
{
    if (!c || !rhs_dev || !p_dev || max_cycles < 0 || !aligned16(rhs_dev, p_dev)) return PS_EINVAL;
    if (!c->have_coef || !c->mg_ready) return PS_ESTATE;
    for (ps_ctx *k = c->child; k; k = k->child) k->stream = c->stream;
    int cyc = 0, converged = 0, rc = 0;
    // Safeguard M7: the parameters of this call; omega_c is lowered by
    // omega_c_step (never below 1) once stall_cycles cycles in a row have ended with a norm that
    // is not below the best so far.  Same bookkeeping, in the same order, as the oracle's loop.
    ps_mg_params q = c->mgp;
    double best = 0.0;
    int have_best = 0, stall = 0;
    auto safeguard = [&](double rr) {
        if (q.stall_cycles <= 0) return;
        if (!have_best || rr < best) {
            best = rr; have_best = 1; stall = 0;
        } else if (++stall >= q.stall_cycles) {
            q.omega_c = q.omega_c - q.omega_c_step;
            if (q.omega_c < 1.0) q.omega_c = 1.0;
            best = rr; stall = 0;
        }
    };
    if (mg_fused_norm_ok(c) && max_cycles > 0) {
        // (cycle, check)* as below, but the check of cycle n rides on the residual + restriction
        // pass that opens cycle n + 1 (one pass of 41 B/cell instead of 40 + 41); the pass after
        // the last cycle only serves the norm
        for (cyc = 0;; ++cyc) {
            if ((rc = mg_launch_residual_restrict_norm(c, rhs_dev, p_dev, c->child->lv_rhs)))
                return rc;
            if (cyc >= 1) {
                PS_CUDA(cudaStreamSynchronize(c->stream));
                if (tol > 0.0 && c->h_scal[1] <= tol) { converged = 1; break; }
                if (cyc == max_cycles || !std::isfinite(c->h_scal[1])) break;
                safeguard(c->h_scal[1]);
            }
            if ((rc = mg_cycle(c, q, rhs_dev, p_dev, 0, true))) return rc;
        }
        if (info) {
            info->sweeps = cyc;
            info->converged = converged;
            info->res_abs = c->h_scal[0];
            info->res_rel = c->h_scal[1];
            info->rhs_norm = c->h_scal[2];
        }
        return PS_OK;
    }
    for (cyc = 1; cyc <= max_cycles; ++cyc) {
        if ((rc = mg_cycle(c, q, rhs_dev, p_dev))) return rc;
        if ((rc = enqueue_residual(c, rhs_dev, p_dev))) return rc;
        PS_CUDA(cudaStreamSynchronize(c->stream));
        if (tol > 0.0 && c->h_scal[1] <= tol) { converged = 1; break; }
        if (!std::isfinite(c->h_scal[1])) break;
        safeguard(c->h_scal[1]);
    }
    if (cyc > max_cycles) cyc = max_cycles;
    if (max_cycles == 0) {
        if ((rc = enqueue_residual(c, rhs_dev, p_dev))) return rc;
        PS_CUDA(cudaStreamSynchronize(c->stream));
    }
    if (info) {
        info->sweeps = cyc;
        info->converged = converged;
        info->res_abs = c->h_scal[0];
        info->res_rel = c->h_scal[1];
        info->rhs_norm = c->h_scal[2];
    }
    return PS_OK;
}

int ps_mg_export_coarse(ps_ctx *c, int level, double *ax_dev, double *ay_dev, double *az_dev)
{
    if (!c || level < 0) return PS_EINVAL;
    if (!c->mg_ready) return PS_ESTATE;
    if (level >= c->mg_nlev) return PS_EINVAL;
    ps_ctx *k = c;
    for (int l = 0; l < level; ++l) k = k->child;
    k->stream = c->stream;
    return ps_export_coefficients(k, ax_dev, ay_dev, az_dev);
}

int ps_mg_residual_restrict(ps_ctx *c, const double *rhs_dev, const double *p_dev, double *rc_dev)
{
    if (!c || !rhs_dev || !p_dev || !rc_dev || !aligned16(rhs_dev, p_dev)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    if (c->g.nx % 2 || c->g.ny % 2 || c->g.nz % 2) return PS_EINVAL;
    return mg_launch_residual_restrict(c, rhs_dev, p_dev, rc_dev);
}

int ps_mg_prolong_add(ps_ctx *c, const double *ec_dev, double *p_dev)
{
    if (!c || !ec_dev || !p_dev || !aligned16(p_dev)) return PS_EINVAL;
    if (c->g.nx % 2 || c->g.ny % 2 || c->g.nz % 2) return PS_EINVAL;
    return mg_launch_prolong_add(c, ec_dev, p_dev);
}

}  // extern "C"

extern "C" {

int ps_rhs_from_velocity(ps_ctx *c, const double *ux_dev, const double *uy_dev,
                         const double *uz_dev, double dt, double *rhs_dev)
{
    if (!c || !ux_dev || !uy_dev || !uz_dev || !rhs_dev) return PS_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return PS_EINVAL;
    if (!aligned16(ux_dev, uy_dev, uz_dev, rhs_dev)) return PS_EINVAL;
    const ps::Spacing h{c->dx, c->dy, c->dz};
    int kz = 0;
    if (c->g.nx % 2 == 0 && c->g.ny <= 65535 * ps::ZS_TY) {
        const dim3 grid = zs_grid(c, 32, &kz);
        ps::ps_rhs_from_velocity_pair_kernel<<<grid, ps::ZS_TX * ps::ZS_TY, 0, c->stream>>>(
            c->g, h, ux_dev, uy_dev, uz_dev, dt, rhs_dev, kz);
    } else
        ps::ps_rhs_from_velocity_kernel<<<grid_for(c, c->g.cells(), 256), 256, 0, c->stream>>>(
            c->g, h, ux_dev, uy_dev, uz_dev, dt, rhs_dev);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

int ps_correct_velocity(ps_ctx *c, const double *p_dev, double dt, double *ux_dev, double *uy_dev,
                        double *uz_dev)
{
    if (!c || !p_dev || !ux_dev || !uy_dev || !uz_dev) return PS_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return PS_EINVAL;
    if (!aligned16(p_dev, ux_dev, uy_dev, uz_dev)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    const ps::Spacing h{c->dx, c->dy, c->dz};
    ps::ps_correct_velocity_kernel<<<grid_for(c, c->g.cells(), 256), 256, 0, c->stream>>>(
        c->g, h, c->ax, c->ay, c->az, p_dev, dt, ux_dev, uy_dev, uz_dev);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

int ps_face_divergence(ps_ctx *c, const double *ux_dev, const double *uy_dev, const double *uz_dev,
                       const double *p_dev, double dt, double *div_dev)
{
    if (!c || !ux_dev || !uy_dev || !uz_dev || !p_dev || !div_dev) return PS_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return PS_EINVAL;
    if (!aligned16(ux_dev, uy_dev, uz_dev, p_dev) || !aligned16(div_dev)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    const ps::Spacing h{c->dx, c->dy, c->dz};
    int kz = 0;
    if (c->g.nx % 2 == 0 && c->g.ny <= 65535 * ps::ZS_TY) {
        const dim3 grid = zs_grid(c, 8, &kz);
        ps::ps_face_divergence_pair_kernel<<<grid, ps::ZS_TX * ps::ZS_TY, 0, c->stream>>>(
            c->g, h, c->ax, c->ay, c->az, ux_dev, uy_dev, uz_dev, p_dev, dt, div_dev, kz);
    } else
        ps::ps_face_divergence_kernel<<<grid_for(c, c->g.cells(), 256), 256, 0, c->stream>>>(
            c->g, h, c->ax, c->ay, c->az, ux_dev, uy_dev, uz_dev, p_dev, dt, div_dev);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

int ps_ssf_rhs(ps_ctx *c, const double *F_dev, const double *kappa_dev, double sigma,
               double *rhs_dev)
{
    if (!c || !F_dev || !kappa_dev || !rhs_dev || !std::isfinite(sigma)) return PS_EINVAL;
    if (!aligned16(F_dev, kappa_dev, rhs_dev)) return PS_EINVAL;
    if (!c->have_coef) return PS_ESTATE;
    if (c->g.nx % 2 == 0)
        ps::ps_ssf_rhs_pair_kernel<<<grid_for(c, c->g.cells() / 2, 256), 256, 0, c->stream>>>(
            c->g, c->ax, c->ay, c->az, F_dev, kappa_dev, sigma, rhs_dev);
    else
        ps::ps_ssf_rhs_kernel<<<grid_for(c, c->g.cells(), 256), 256, 0, c->stream>>>(
            c->g, c->ax, c->ay, c->az, F_dev, kappa_dev, sigma, rhs_dev);
    c->launches++;
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

int ps_stream_probe(const double *in_dev, double *out_dev, size_t n, int reads, int blocks,
                    void *cuda_stream)
{
    if (!in_dev || !out_dev || n < 2 || (n & 1) || blocks < 1 || !aligned16(in_dev, out_dev))
        return PS_EINVAL;
    const double2 *in = reinterpret_cast<const double2 *>(in_dev);
    double2 *out = reinterpret_cast<double2 *>(out_dev);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    switch (reads) {
        case 1: ps::ps_stream_probe_kernel<1><<<blocks, 512, 0, st>>>(in, out, n / 2); break;
        case 3: ps::ps_stream_probe_kernel<3><<<blocks, 512, 0, st>>>(in, out, n / 2); break;
        case 5: ps::ps_stream_probe_kernel<5><<<blocks, 512, 0, st>>>(in, out, n / 2); break;
        default: return PS_EINVAL;
    }
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}

const char *ps_strerror(int code)
{
    switch (code) {
        case PS_OK: return "ok";
        case PS_EINVAL: return "invalid argument";
        case PS_ESTATE: return "coefficients not set: call ps_set_fraction first";
        case PS_ECUDA: return g_cuda_msg;
        case PS_ENOMEM: return "out of memory";
        case PS_ETOOBIG:
            return "grid too large for ps_residual_noalloc: more than PS_NOALLOC_MAX_CELLS "
                   "(268435456) cells do not fit its fixed in-library scratch array";
        default: return "unknown error code";
    }
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// ps_residual_noalloc: the residual norms for callers that must not allocate (see the header).
//
// ps_residual needs scratch memory beyond its inputs and outputs: one pair of partial sums per
// 4096-cell chunk, which the final pass adds up.  It takes them from the context's workspace,
// which somebody had to allocate.  The variant below keeps them in an array that is part of the
// library image instead: every GPU that loads the library carries these 1 MiB + 256 B from the
// moment the module is loaded until the process exits, and no call ever allocates or frees.
namespace {

constexpr int PS_NA_MAX_PARTS = (int)(PS_NOALLOC_MAX_CELLS / ps::RED_CHUNK);   // 65,536 chunks
static_assert((long long)PS_NA_MAX_PARTS * ps::RED_CHUNK == PS_NOALLOC_MAX_CELLS, "whole chunks");
constexpr int PS_NA_TAIL = 32;   // 256 bytes behind the partials; word 0 is the ticket counter

// [0, MAX_PARTS): sum r^2 per chunk; [MAX_PARTS, 2 MAX_PARTS): sum rhs^2 per chunk; then the
// ticket counter (blocks of the running call that have delivered their pair).  Shared by every
// call on this device; holds whatever the last call left.
static __device__ __align__(256) double ps_na_scratch[2 * PS_NA_MAX_PARTS + PS_NA_TAIL];

// In host code `ps_na_scratch` is only a handle for the runtime, not an address a kernel could
// use; the device address is asked for once per device and kept here.
constexpr int PS_NA_MAX_DEVICES = 64;
std::atomic<double *> g_na_scratch_dev[PS_NA_MAX_DEVICES];

// One launch instead of ps_residual's two: every block reduces its chunk exactly as
// ps_residual_partial(_pair)_kernel does and stores the pair in the scratch array; the block that
// draws the last ticket then adds the pairs up in the order of ps_reduce_final_kernel (its 1024
// threads and 32 warps are walked through by the 256 threads and 8 warps here), so the three
// numbers are bitwise those of ps_residual.
template <bool PAIR>
__global__ void __launch_bounds__(ps::RED_THREADS)
ps_residual_noalloc_kernel(ps::Grid g, const double *__restrict__ ax,
                           const double *__restrict__ ay, const double *__restrict__ az,
                           const double *__restrict__ rhs, const double *__restrict__ p,
                           double *scratch, double *__restrict__ out)
{
    __shared__ double sm[2 * ps::FIN_THREADS / 32];
    __shared__ int am_last;
    double *partR2 = scratch, *partB2 = scratch + PS_NA_MAX_PARTS;
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch + 2 * PS_NA_MAX_PARTS);
    const size_t N = g.cells();
    const size_t base = (size_t)blockIdx.x * ps::RED_CHUNK;
    double r2 = 0.0, b2 = 0.0;
    if (PAIR) {
#pragma unroll 2
        for (int m = 0; m < ps::RED_CHUNK / (2 * ps::RED_THREADS); ++m) {
            const size_t n = base + 2 * ((size_t)m * ps::RED_THREADS + threadIdx.x);
            if (n < N) {
                const int i = (int)((unsigned)n % (unsigned)g.nx);
                const unsigned t = (unsigned)n / (unsigned)g.nx;
                const int j = (int)(t % (unsigned)g.ny);
                const int k = (int)(t / (unsigned)g.ny);
                double2 b;
                const double2 r = ps::residual_pair(g, ax, ay, az, rhs, p, i, j, k, n, b);
                r2 = r2 + r.x * r.x;
                r2 = r2 + r.y * r.y;
                b2 = b2 + b.x * b.x;
                b2 = b2 + b.y * b.y;
            }
        }
    } else {
#pragma unroll 4
        for (int m = 0; m < ps::RED_CHUNK / ps::RED_THREADS; ++m) {
            const size_t n = base + (size_t)m * ps::RED_THREADS + threadIdx.x;
            if (n < N) {
                const int i = (int)((unsigned)n % (unsigned)g.nx);
                const unsigned t = (unsigned)n / (unsigned)g.nx;
                const int j = (int)(t % (unsigned)g.ny);
                const int k = (int)(t / (unsigned)g.ny);
                const ps::Stencil s = ps::gather(g, ax, ay, az, p, i, j, k, n);
                const double b = rhs[n];
                const double r = ps::residual_at(s.axm, s.axp, s.aym, s.ayp, s.azm, s.azp, s.pxm,
                                                 s.pxp, s.pym, s.pyp, s.pzm, s.pzp, p[n], b);
                r2 = r2 + r * r;
                b2 = b2 + b * b;
            }
        }
    }
    const double Rs = ps::block_tree_sum<ps::RED_THREADS>(r2, sm);
    const double Bs = ps::block_tree_sum<ps::RED_THREADS>(b2, sm);
    if (threadIdx.x == 0) {
        __stcg(partR2 + blockIdx.x, Rs);
        __stcg(partB2 + blockIdx.x, Bs);
        __threadfence();                                  // the pair is visible before the ticket
        am_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!am_last) return;
    __threadfence();                                      // every other block's pair is visible now
    const int nparts = (int)gridDim.x;
    const int lane = threadIdx.x & 31;
    double *smR = sm, *smB = sm + ps::FIN_THREADS / 32;
    for (int vw = threadIdx.x >> 5; vw < ps::FIN_THREADS / 32; vw += ps::RED_THREADS / 32) {
        double fr = 0.0, fb = 0.0;
        for (int q = vw * 32 + lane; q < nparts; q += ps::FIN_THREADS) {
            fr = fr + __ldcg(partR2 + q);
            fb = fb + __ldcg(partB2 + q);
        }
        fr = ps::warp_tree_sum(fr);
        fb = ps::warp_tree_sum(fb);
        if (lane == 0) { smR[vw] = fr; smB[vw] = fb; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double R = 0.0, B = 0.0;
#pragma unroll
        for (int q = 0; q < ps::FIN_THREADS / 32; ++q) R = R + smR[q];
#pragma unroll
        for (int q = 0; q < ps::FIN_THREADS / 32; ++q) B = B + smB[q];
        const double ra = sqrt(R), bn = sqrt(B);
        out[0] = ra;
        out[1] = (bn > 0.0) ? ra / bn : ra;
        out[2] = bn;
    }
}

}  // namespace

extern "C" int ps_residual_noalloc(int nx, int ny, int nz, const double *ax_dev,
                                   const double *ay_dev, const double *az_dev,
                                   const double *rhs_dev, const double *p_dev, void *cuda_stream,
                                   double *out_dev)
{
    if (nx < 1 || ny < 1 || nz < 2 || (nz & 1)) return PS_EINVAL;
    if (!ax_dev || !ay_dev || !az_dev || !rhs_dev || !p_dev || !out_dev) return PS_EINVAL;
    if (!aligned16(ax_dev, ay_dev, az_dev) || !aligned16(rhs_dev, p_dev) ||
        ((uintptr_t)out_dev & 7u) != 0)
        return PS_EINVAL;
    if ((double)nx * (double)ny * (double)nz > (double)PS_NOALLOC_MAX_CELLS) return PS_ETOOBIG;
    const ps::Grid g{nx, ny, nz};
    int dev = -1;
    PS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= PS_NA_MAX_DEVICES) return PS_EINVAL;
    // Set-up, once per device, with that device current: the device address of the array.
    double *scratch = g_na_scratch_dev[dev].load(std::memory_order_acquire);
    if (!scratch) {
        PS_CUDA(cudaGetSymbolAddress((void **)&scratch, ps_na_scratch));
        g_na_scratch_dev[dev].store(scratch, std::memory_order_release);
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The ticket counter must start at zero; the partials need no clearing (every slot the final
    // pass reads is written by this launch first).  A memset node, not an allocation.
    PS_CUDA(cudaMemsetAsync(scratch + 2 * PS_NA_MAX_PARTS, 0, PS_NA_TAIL * sizeof(double), st));
    const int nparts = nparts_for(g.cells());
    if (nx % 2 == 0)
        ps_residual_noalloc_kernel<true><<<nparts, ps::RED_THREADS, 0, st>>>(
            g, ax_dev, ay_dev, az_dev, rhs_dev, p_dev, scratch, out_dev);
    else
        ps_residual_noalloc_kernel<false><<<nparts, ps::RED_THREADS, 0, st>>>(
            g, ax_dev, ay_dev, az_dev, rhs_dev, p_dev, scratch, out_dev);
    PS_CUDA(cudaGetLastError());
    return PS_OK;
}
