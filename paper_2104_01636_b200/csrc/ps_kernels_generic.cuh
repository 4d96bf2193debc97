// ps_kernels_generic.cuh -- shape-generic CUDA kernels of the pressure-Poisson path (sm_100a).
//
//   ps_coef_build_kernel      F -> rho -> ax, ay, az           PAPER.md:66 eq (4), :92, :117, :195
//   ps_half_sweep_kernel      one colour of red-black SOR
//   ps_residual_partial_kernel / ps_reduce_final_kernel         DESIGN.md reading S5 (paper silent)
//
// These work for any nx, ny >= 1 and even nz >= 2 and are the reference schedule of the CUDA
// path: one thread per cell (coefficients, residual) or per cell of the active colour (sweep),
// plain coalesced global loads, neighbour reuse left to L1/L2.  The fast kernels of
// ps_kernels_zmarch.cuh and ps_kernels_resident.cuh compute the same expressions in the same
// order, so every variant gives bitwise identical p.  Compile with --fmad=false: every * and + below rounds separately.
#pragma once
#include <cstddef>
#include <cstdint>

namespace ps {

struct Grid {
    int nx, ny, nz;
    __host__ __device__ size_t cells() const { return (size_t)nx * (size_t)ny * (size_t)nz; }
    __host__ __device__ size_t idx(int i, int j, int k) const {
        return (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
    }
};

// One SOR update written once, used by every kernel variant.  Argument order = summation order.
//   s = sum_f a_f p_nb (12 roundings, left to right), d = sum_f a_f, g = (s - rhs)/d,
//   p <- p + omega (g - p).
__device__ __forceinline__ double sor_update(double axm, double axp, double aym, double ayp,
                                             double azm, double azp, double pxm, double pxp,
                                             double pym, double pyp, double pzm, double pzp,
                                             double pc, double rhs, double omega)
{
    const double s = ((((axm * pxm + axp * pxp) + aym * pym) + ayp * pyp) + azm * pzm) + azp * pzp;
    const double d = ((((axm + axp) + aym) + ayp) + azm) + azp;
    const double g = (s - rhs) / d;
    return pc + omega * (g - pc);
}

// r_c = rhs_c - (s - d p_c), same s and d.
__device__ __forceinline__ double residual_at(double axm, double axp, double aym, double ayp,
                                              double azm, double azp, double pxm, double pxp,
                                              double pym, double pyp, double pzm, double pzp,
                                              double pc, double rhs)
{
    const double s = ((((axm * pxm + axp * pxp) + aym * pym) + ayp * pyp) + azm * pzm) + azp * pzp;
    const double d = ((((axm + axp) + aym) + ayp) + azm) + azp;
    return rhs - (s - d * pc);
}

// ---------------------------------------------------------------------------------------------
// Coefficient build: one thread per cell, 8 B in (plus neighbour reads served by L1/L2), 24 B out.
__global__ void __launch_bounds__(256)
ps_coef_build_kernel(Grid g, double cx, double cy, double cz, double rho_l, double rho_g,
                     const double *__restrict__ F, double *__restrict__ ax,
                     double *__restrict__ ay, double *__restrict__ az)
{
    const size_t N = g.cells();
    const size_t plane = (size_t)g.nx * g.ny;
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < N;
         n += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)((unsigned)n % (unsigned)g.nx);
        const unsigned t = (unsigned)n / (unsigned)g.nx;
        const int j = (int)(t % (unsigned)g.ny);
        const int k = (int)(t / (unsigned)g.ny);
        const double Fc = F[n];
        const double rc = (rho_l * Fc) + (rho_g * (1.0 - Fc));
        double vx = 0.0, vy = 0.0;
        if (i < g.nx - 1) {
            const double Fn = F[n + 1];
            const double rn = (rho_l * Fn) + (rho_g * (1.0 - Fn));
            vx = cx / (0.5 * (rc + rn));
        }
        if (j < g.ny - 1) {
            const double Fn = F[n + g.nx];
            const double rn = (rho_l * Fn) + (rho_g * (1.0 - Fn));
            vy = cy / (0.5 * (rc + rn));
        }
        const size_t nz_up = (k + 1 < g.nz) ? n + plane : n - plane * (size_t)(g.nz - 1);
        const double Fz = F[nz_up];
        const double rz = (rho_l * Fz) + (rho_g * (1.0 - Fz));
        ax[n] = vx;
        ay[n] = vy;
        az[n] = cz / (0.5 * (rc + rz));
    }
}

// The same for even nx: one thread per x-pair of cells, 16-byte loads and stores, six independent
// divisions in flight per thread.  Same expressions, same values.
__global__ void __launch_bounds__(256)
ps_coef_build_pair_kernel(Grid g, double cx, double cy, double cz, double rho_l, double rho_g,
                          const double *__restrict__ F, double *__restrict__ ax,
                          double *__restrict__ ay, double *__restrict__ az)
{
    const unsigned hx = (unsigned)g.nx >> 1;
    const unsigned pairs = hx * (unsigned)g.ny * (unsigned)g.nz;
    const size_t plane = (size_t)g.nx * g.ny;
    for (unsigned h = blockIdx.x * blockDim.x + threadIdx.x; h < pairs; h += gridDim.x * blockDim.x) {
        const int i = 2 * (int)(h % hx);
        const unsigned t = h / hx;
        const int j = (int)(t % (unsigned)g.ny), k = (int)(t / (unsigned)g.ny);
        const size_t n = g.idx(i, j, k);
        const size_t nzp = (k + 1 < g.nz) ? n + plane : n - plane * (size_t)(g.nz - 1);
        const double2 Fc = *reinterpret_cast<const double2 *>(F + n);
        const double2 Fz = *reinterpret_cast<const double2 *>(F + nzp);
        const double r0 = (rho_l * Fc.x) + (rho_g * (1.0 - Fc.x));
        const double r1 = (rho_l * Fc.y) + (rho_g * (1.0 - Fc.y));
        double2 vx, vy = make_double2(0.0, 0.0), vz;
        vx.x = cx / (0.5 * (r0 + r1));
        vx.y = 0.0;
        if (i + 2 < g.nx) {
            const double Fn = F[n + 2];
            vx.y = cx / (0.5 * (r1 + ((rho_l * Fn) + (rho_g * (1.0 - Fn)))));
        }
        if (j < g.ny - 1) {
            const double2 Fy = *reinterpret_cast<const double2 *>(F + n + g.nx);
            vy.x = cy / (0.5 * (r0 + ((rho_l * Fy.x) + (rho_g * (1.0 - Fy.x)))));
            vy.y = cy / (0.5 * (r1 + ((rho_l * Fy.y) + (rho_g * (1.0 - Fy.y)))));
        }
        vz.x = cz / (0.5 * (r0 + ((rho_l * Fz.x) + (rho_g * (1.0 - Fz.x)))));
        vz.y = cz / (0.5 * (r1 + ((rho_l * Fz.y) + (rho_g * (1.0 - Fz.y)))));
        *reinterpret_cast<double2 *>(ax + n) = vx;
        *reinterpret_cast<double2 *>(ay + n) = vy;
        *reinterpret_cast<double2 *>(az + n) = vz;
    }
}

// O1 alone: rho = rho_l F + rho_g (1 - F), kept for the sweep variant that rebuilds the face
// coefficients on the fly (PS_KERNEL_FUSED_OTF).  8 B in, 8 B out per cell.
__global__ void __launch_bounds__(256)
ps_rho_build_kernel(size_t N, double rho_l, double rho_g, const double *__restrict__ F,
                    double *__restrict__ rho)
{
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < N;
         n += (size_t)gridDim.x * blockDim.x) {
        const double Fc = F[n];
        rho[n] = (rho_l * Fc) + (rho_g * (1.0 - Fc));
    }
}

// ---------------------------------------------------------------------------------------------
// Gather the six coefficients and neighbour values of cell (i,j,k) from natural-layout arrays.
// Wall neighbours are read at the clamped index (a finite number) and meet a 0.0 coefficient.
struct Stencil {
    double axm, axp, aym, ayp, azm, azp, pxm, pxp, pym, pyp, pzm, pzp;
};

__device__ __forceinline__ Stencil gather(const Grid &g, const double *__restrict__ ax,
                                          const double *__restrict__ ay,
                                          const double *__restrict__ az, const double *p, int i,
                                          int j, int k, size_t n)
{
    const size_t plane = (size_t)g.nx * g.ny;
    const size_t nzm = (k > 0) ? n - plane : n + plane * (size_t)(g.nz - 1);
    const size_t nzp = (k + 1 < g.nz) ? n + plane : n - plane * (size_t)(g.nz - 1);
    Stencil s;
    s.axm = (i > 0) ? ax[n - 1] : 0.0;
    s.axp = ax[n];
    s.aym = (j > 0) ? ay[n - g.nx] : 0.0;
    s.ayp = ay[n];
    s.azm = az[nzm];
    s.azp = az[n];
    s.pxm = p[(i > 0) ? n - 1 : n];
    s.pxp = p[(i < g.nx - 1) ? n + 1 : n];
    s.pym = p[(j > 0) ? n - g.nx : n];
    s.pyp = p[(j < g.ny - 1) ? n + g.nx : n];
    s.pzm = p[nzm];
    s.pzp = p[nzp];
    return s;
}

// Residuals of the x-pair of cells (n, n+1) (n even, nx even) with 16-byte loads; R returns the
// rhs pair.  Same expression as residual_at(gather(...)) for each of the two cells.
__device__ __forceinline__ double2 ld2(const double *q)
{
    return *reinterpret_cast<const double2 *>(q);
}

__device__ __forceinline__ double2 residual_pair(const Grid &g, const double *__restrict__ ax,
                                                 const double *__restrict__ ay,
                                                 const double *__restrict__ az,
                                                 const double *__restrict__ rhs,
                                                 const double *__restrict__ p, int i, int j, int k,
                                                 size_t n, double2 &R)
{
    const size_t plane = (size_t)g.nx * g.ny;
    const size_t nzm = (k > 0) ? n - plane : n + plane * (size_t)(g.nz - 1);
    const size_t nzp = (k + 1 < g.nz) ? n + plane : n - plane * (size_t)(g.nz - 1);
    const double2 P = ld2(p + n), AX = ld2(ax + n), AY = ld2(ay + n), AZ = ld2(az + n);
    R = ld2(rhs + n);
    const double axl = (i > 0) ? ax[n - 1] : 0.0;
    const double2 AYm = (j > 0) ? ld2(ay + n - g.nx) : make_double2(0.0, 0.0);
    const double2 AZm = ld2(az + nzm);
    const double pl = p[(i > 0) ? n - 1 : n];
    const double pr = p[(i + 2 < g.nx) ? n + 2 : n + 1];
    const double2 Pym = ld2(p + ((j > 0) ? n - g.nx : n));
    const double2 Pyp = ld2(p + ((j < g.ny - 1) ? n + g.nx : n));
    const double2 Pzm = ld2(p + nzm), Pzp = ld2(p + nzp);
    double2 r;
    r.x = residual_at(axl, AX.x, AYm.x, AY.x, AZm.x, AZ.x, pl, P.y, Pym.x, Pyp.x, Pzm.x, Pzp.x, P.x,
                      R.x);
    r.y = residual_at(AX.x, AX.y, AYm.y, AY.y, AZm.y, AZ.y, P.x, pr, Pym.y, Pyp.y, Pzm.y, Pzp.y, P.y,
                      R.y);
    return r;
}

// Half-sweep, in place: one thread per cell of the active colour ((i+j+k)&1 == colour).
// Cells of one colour never read each other, so no ordering between threads is needed.
__global__ void __launch_bounds__(256)
ps_half_sweep_kernel(Grid g, const double *__restrict__ ax, const double *__restrict__ ay,
                     const double *__restrict__ az, const double *__restrict__ rhs, double *p,
                     double omega, int colour)
{
    const int hx = (g.nx + 1) >> 1;
    const size_t total = (size_t)hx * g.ny * g.nz;
    for (size_t h = (size_t)blockIdx.x * blockDim.x + threadIdx.x; h < total;
         h += (size_t)gridDim.x * blockDim.x) {
        const int ih = (int)((unsigned)h % (unsigned)hx);
        const unsigned t = (unsigned)h / (unsigned)hx;
        const int j = (int)(t % (unsigned)g.ny);
        const int k = (int)(t / (unsigned)g.ny);
        const int i = 2 * ih + ((j + k + colour) & 1);
        if (i >= g.nx) continue;
        const size_t n = g.idx(i, j, k);
        const Stencil s = gather(g, ax, ay, az, p, i, j, k, n);
        p[n] = sor_update(s.axm, s.axp, s.aym, s.ayp, s.azm, s.azp, s.pxm, s.pxp, s.pym, s.pyp,
                          s.pzm, s.pzp, p[n], rhs[n], omega);
    }
}

// ---------------------------------------------------------------------------------------------
// Deterministic two-pass reduction.  Pass 1: block b owns cells [b*CHUNK, (b+1)*CHUNK); thread t
// adds its cells t, t+256, ... in that order, then a fixed xor-shuffle tree per warp and a fixed
// left-to-right sum over the 8 warps.  The partition depends on N only (not on the SM count), so
// the result is reproducible across devices and launches.  No floating-point atomics.
constexpr int RED_THREADS = 256;
constexpr int RED_CHUNK = 4096;

__device__ __forceinline__ double warp_tree_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = v + __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <int THREADS>
__device__ __forceinline__ double block_tree_sum(double v, double *smem /* THREADS/32 */)
{
    v = warp_tree_sum(v);
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) smem[w] = v;
    __syncthreads();
    double tot = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < THREADS / 32; ++q) tot = tot + smem[q];
    }
    __syncthreads();
    return tot;   // valid on thread 0
}

__global__ void __launch_bounds__(RED_THREADS)
ps_residual_partial_kernel(Grid g, const double *__restrict__ ax, const double *__restrict__ ay,
                           const double *__restrict__ az, const double *__restrict__ rhs,
                           const double *__restrict__ p, double *__restrict__ partR2,
                           double *__restrict__ partB2)
{
    __shared__ double sm[RED_THREADS / 32];
    const size_t N = g.cells();
    const size_t base = (size_t)blockIdx.x * RED_CHUNK;
    double r2 = 0.0, b2 = 0.0;
#pragma unroll 4
    for (int m = 0; m < RED_CHUNK / RED_THREADS; ++m) {
        const size_t n = base + (size_t)m * RED_THREADS + threadIdx.x;
        if (n < N) {
            const int i = (int)((unsigned)n % (unsigned)g.nx);
            const unsigned t = (unsigned)n / (unsigned)g.nx;
            const int j = (int)(t % (unsigned)g.ny);
            const int k = (int)(t / (unsigned)g.ny);
            const Stencil s = gather(g, ax, ay, az, p, i, j, k, n);
            const double b = rhs[n];
            const double r = residual_at(s.axm, s.axp, s.aym, s.ayp, s.azm, s.azp, s.pxm, s.pxp,
                                         s.pym, s.pyp, s.pzm, s.pzp, p[n], b);
            r2 = r2 + r * r;
            b2 = b2 + b * b;
        }
    }
    const double R = block_tree_sum<RED_THREADS>(r2, sm);
    const double B = block_tree_sum<RED_THREADS>(b2, sm);
    if (threadIdx.x == 0) {
        partR2[blockIdx.x] = R;
        partB2[blockIdx.x] = B;
    }
}

// The same for even nx (every ABI pointer is 16-byte aligned): thread t takes the x-pairs t, t+256, ... of the
// block's chunk (left cell first).  A different but equally fixed summation tree.
__global__ void __launch_bounds__(RED_THREADS)
ps_residual_partial_pair_kernel(Grid g, const double *__restrict__ ax,
                                const double *__restrict__ ay, const double *__restrict__ az,
                                const double *__restrict__ rhs, const double *__restrict__ p,
                                double *__restrict__ partR2, double *__restrict__ partB2)
{
    __shared__ double sm[RED_THREADS / 32];
    const size_t N = g.cells();
    const size_t base = (size_t)blockIdx.x * RED_CHUNK;
    double r2 = 0.0, b2 = 0.0;
#pragma unroll 2
    for (int m = 0; m < RED_CHUNK / (2 * RED_THREADS); ++m) {
        const size_t n = base + 2 * ((size_t)m * RED_THREADS + threadIdx.x);
        if (n < N) {
            const int i = (int)((unsigned)n % (unsigned)g.nx);
            const unsigned t = (unsigned)n / (unsigned)g.nx;
            const int j = (int)(t % (unsigned)g.ny);
            const int k = (int)(t / (unsigned)g.ny);
            double2 b;
            const double2 r = residual_pair(g, ax, ay, az, rhs, p, i, j, k, n, b);
            r2 = r2 + r.x * r.x;
            r2 = r2 + r.y * r.y;
            b2 = b2 + b.x * b.x;
            b2 = b2 + b.y * b.y;
        }
    }
    const double Rs = block_tree_sum<RED_THREADS>(r2, sm);
    const double Bs = block_tree_sum<RED_THREADS>(b2, sm);
    if (threadIdx.x == 0) {
        partR2[blockIdx.x] = Rs;
        partB2[blockIdx.x] = Bs;
    }
}

// Pass 2: one block; thread t adds partials t, t+1024, ... in order, then the same fixed tree.
// out[0] = ||r||_2, out[1] = ||r||_2/||rhs||_2 (||r||_2 if rhs == 0), out[2] = ||rhs||_2.
constexpr int FIN_THREADS = 1024;

__global__ void __launch_bounds__(FIN_THREADS)
ps_reduce_final_kernel(const double *__restrict__ partR2, const double *__restrict__ partB2,
                       int nparts, double *__restrict__ out)
{
    __shared__ double sm[FIN_THREADS / 32];
    double r2 = 0.0, b2 = 0.0;
    for (int q = threadIdx.x; q < nparts; q += FIN_THREADS) {
        r2 = r2 + partR2[q];
        b2 = b2 + partB2[q];
    }
    const double R = block_tree_sum<FIN_THREADS>(r2, sm);
    const double B = block_tree_sum<FIN_THREADS>(b2, sm);
    if (threadIdx.x == 0) {
        const double ra = sqrt(R), bn = sqrt(B);
        const double rr = (bn > 0.0) ? ra / bn : ra;
        out[0] = ra;
        out[1] = rr;
        out[2] = bn;
    }
}

// ---------------------------------------------------------------------------------------------
// Bandwidth probe with the sweep's read:write mix (bench.py's second roofline denominator): out =
// sum of READS input streams, 16-byte accesses, two elements of every stream in flight per
// thread.  The fused sweep reads five streams (p, ax, ay, az, rhs) and writes one; a device copy
// (the MEASURED_PEAKS.json figure) reads one and writes one, and HBM turns around between reads and
// writes less often in the first case.  No part of the solve path.
template <int READS>
__global__ void __launch_bounds__(512)
ps_stream_probe_kernel(const double2 *__restrict__ in, double2 *__restrict__ out, size_t n2)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; q + stride < n2; q += 2 * stride) {
        double2 a[READS], b[READS];
#pragma unroll
        for (int r = 0; r < READS; ++r) {
            a[r] = __ldcs(in + (size_t)r * n2 + q);
            b[r] = __ldcs(in + (size_t)r * n2 + q + stride);
        }
        double2 sa = a[0], sb = b[0];
#pragma unroll
        for (int r = 1; r < READS; ++r) {
            sa.x = sa.x + a[r].x; sa.y = sa.y + a[r].y;
            sb.x = sb.x + b[r].x; sb.y = sb.y + b[r].y;
        }
        __stcs(out + q, sa);
        __stcs(out + q + stride, sb);
    }
    if (q < n2) {
        double2 sa = __ldcs(in + q);
#pragma unroll
        for (int r = 1; r < READS; ++r) {
            const double2 v = __ldcs(in + (size_t)r * n2 + q);
            sa.x = sa.x + v.x; sa.y = sa.y + v.y;
        }
        __stcs(out + q, sa);
    }
}

}  // namespace ps
