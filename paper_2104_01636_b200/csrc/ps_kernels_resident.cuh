// ps_kernels_resident.cuh -- many red-black SOR sweeps in ONE launch for grids that live in L2.
//
// The small grids (BASELINE.json configs 1-2; the coarse levels of the multigrid hierarchy) are
// bound by launch and pipeline start-up latency, not by HBM: a sweep moves at most a few MB.  This
// kernel is launched cooperatively (co-residency guaranteed) with at most one CTA per SM and runs
// `nsweeps` sweeps in place, one grid-wide barrier after every half-sweep (cells of one colour
// never read each other, so a half-sweep needs no ordering inside).  The barrier is a monotonic
// arrival counter in global memory (zeroed by the host before the launch): one atomic per CTA and
// a polling load, about 1 us against 2.4 us of cooperative_groups' grid.sync(); a single-CTA
// launch (<= 1024 cells of a colour) only needs __syncthreads().  Each thread keeps the same cells for the whole launch, so
// the coefficients and rhs it needs stay in its SM's L1; p is read through L2 (ld.global.cg), the
// level at which the writes of the other SMs are coherent.
// Same update expression, same order as every other kernel (sor_update) -> bitwise identical p.
#pragma once
#include "ps_kernels_generic.cuh"

namespace ps {

constexpr int RES_THREADS = 256;        // multi-CTA launches
constexpr int RES_THREADS_ONE = 1024;   // single-CTA launches

__device__ __forceinline__ void res_grid_barrier(unsigned *ctr, unsigned target)
{
    __syncthreads();                    // the CTA's stores precede thread 0's fence
    if (gridDim.x > 1) {
        if (threadIdx.x == 0) {
            __threadfence();
            atomicAdd(ctr, 1u);
            while (*(volatile unsigned *)ctr < target) { }
            __threadfence();
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(RES_THREADS_ONE)
ps_resident_sweeps_kernel(Grid g, const double *__restrict__ ax, const double *__restrict__ ay,
                          const double *__restrict__ az, const double *__restrict__ rhs, double *p,
                          double omega, int nsweeps, unsigned *barrier_ctr)
{
    const int hx = (g.nx + 1) >> 1;
    const size_t total = (size_t)hx * g.ny * g.nz;
    const size_t plane = (size_t)g.nx * g.ny;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int s = 0; s < 2 * nsweeps; ++s) {
        const int colour = s & 1;
        for (size_t h = (size_t)blockIdx.x * blockDim.x + threadIdx.x; h < total; h += stride) {
            const int ih = (int)((unsigned)h % (unsigned)hx);
            const unsigned t = (unsigned)h / (unsigned)hx;
            const int j = (int)(t % (unsigned)g.ny);
            const int k = (int)(t / (unsigned)g.ny);
            const int i = 2 * ih + ((j + k + colour) & 1);
            if (i >= g.nx) continue;
            const size_t n = g.idx(i, j, k);
            const size_t nzm = (k > 0) ? n - plane : n + plane * (size_t)(g.nz - 1);
            const size_t nzp = (k + 1 < g.nz) ? n + plane : n - plane * (size_t)(g.nz - 1);
            const double axm = (i > 0) ? __ldg(ax + n - 1) : 0.0, axp = __ldg(ax + n);
            const double aym = (j > 0) ? __ldg(ay + n - g.nx) : 0.0, ayp = __ldg(ay + n);
            const double azm = __ldg(az + nzm), azp = __ldg(az + n);
            const double pxm = __ldcg(p + ((i > 0) ? n - 1 : n));
            const double pxp = __ldcg(p + ((i < g.nx - 1) ? n + 1 : n));
            const double pym = __ldcg(p + ((j > 0) ? n - g.nx : n));
            const double pyp = __ldcg(p + ((j < g.ny - 1) ? n + g.nx : n));
            const double pzm = __ldcg(p + nzm), pzp = __ldcg(p + nzp);
            const double pc = __ldcg(p + n);
            __stcg(p + n, sor_update(axm, axp, aym, ayp, azm, azp, pxm, pxp, pym, pyp, pzm, pzp, pc,
                                     __ldg(rhs + n), omega));
        }
        res_grid_barrier(barrier_ctr, (unsigned)(s + 1) * gridDim.x);
    }
}

}  // namespace ps
