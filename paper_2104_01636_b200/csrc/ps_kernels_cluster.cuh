// ps_kernels_cluster.cuh -- many red-black SOR sweeps in ONE launch for grids that fit the shared
// memory of one thread-block cluster (sm_100a: up to 16 CTAs x 227 KB).
//
// The smallest grids (BASELINE.json config 1; the coarse levels of the multigrid hierarchy, which
// run 48 sweeps per visit) are bound by synchronisation latency, not by bandwidth: the resident
// kernel (ps_kernels_resident.cuh) spends 2.6 us per half-sweep on a grid-wide barrier through
// global memory and on L2 round trips.  Here the whole problem lives on chip for the launch:
//   * the launch is ONE cluster of C CTAs (C = 16, 8, 4, 2 or 1, the largest that divides nz);
//     CTA r owns the z slab [r nz/C, (r+1) nz/C) and keeps p, ax, ay, rhs of the slab and az of
//     the slab plus the plane below it in shared memory (loaded once, p written back once);
//   * a half-sweep updates the cells of one colour in place in shared memory; the z neighbours
//     of the slab's first and last plane are read from the neighbouring CTA's shared memory
//     (distributed shared memory, periodic in the cluster rank).  Cells of one colour never read
//     each other, so the only ordering needed is one cluster barrier (barrier.cluster
//     arrive.release / wait.acquire, ~0.2 us) per half-sweep.
// Same update expression, same order as every other kernel (sor_update) -> bitwise identical p.
#pragma once
#include <cooperative_groups.h>

#include "ps_kernels_generic.cuh"

namespace ps {

constexpr int CL_THREADS = 1024;
constexpr int CL_ITEMS = 3;            // x-pairs of cells per thread: a slab holds at most 6144 cells
constexpr size_t CL_SMEM_MAX = 227 * 1024;

// shared memory of one CTA: 4 slab fields (p, ax, ay, rhs) + az with one extra plane
inline size_t cl_smem_bytes(const Grid &g, int C)
{
    const size_t plane = (size_t)g.nx * g.ny, pz = (size_t)(g.nz / C);
    return (4 * pz * plane + (pz + 1) * plane) * sizeof(double);
}

// the cluster size for this grid, or 0 if it does not fit
inline int cl_cluster_size(const Grid &g)
{
    for (int C = 16; C >= 1; C >>= 1) {
        if (g.nz % C != 0) continue;
        const size_t pairs = (size_t)((g.nx + 1) / 2) * g.ny * (size_t)(g.nz / C);
        if (cl_smem_bytes(g, C) <= CL_SMEM_MAX && pairs <= (size_t)CL_ITEMS * CL_THREADS) return C;
        return 0;                       // fewer CTAs only need more memory each
    }
    return 0;
}

__global__ void __launch_bounds__(CL_THREADS, 1)
ps_cluster_sweeps_kernel(Grid g, const double *__restrict__ ax, const double *__restrict__ ay,
                         const double *__restrict__ az, const double *__restrict__ rhs, double *p,
                         double omega, int nsweeps)
{
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) double cl_smem[];
    const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int pz = g.nz / C, k0 = rank * pz;
    const int plane = g.nx * g.ny, slab = pz * plane;
    double *P = cl_smem, *AX = P + slab, *AY = AX + slab, *RH = AY + slab, *AZ = RH + slab;
    // AZ: plane 0 = az of the plane below the slab (periodic), planes 1..pz = the slab's own
    const size_t base = (size_t)k0 * plane;
    for (int n = threadIdx.x; n < slab; n += CL_THREADS) {
        P[n] = p[base + n];
        AX[n] = ax[base + n];
        AY[n] = ay[base + n];
        RH[n] = rhs[base + n];
        AZ[plane + n] = az[base + n];
    }
    const size_t below = (size_t)(k0 > 0 ? k0 - 1 : g.nz - 1) * plane;
    for (int n = threadIdx.x; n < plane; n += CL_THREADS) AZ[n] = az[below + n];
    // the slabs of the z neighbours (the CTA itself when the cluster is one CTA: periodic)
    const double *Pdn = cluster.map_shared_rank(P, rank > 0 ? rank - 1 : C - 1);
    const double *Pup = cluster.map_shared_rank(P, rank + 1 < C ? rank + 1 : 0);
    cluster.sync();

    // A thread keeps the same (at most CL_ITEMS) x-pairs of cells for the whole launch -- in each
    // half-sweep it updates the cell of the pair that has the active colour -- so everything that
    // does not depend on the colour is worked out once, here: the index of the pair's left cell,
    // which of its two cells is red, where its six neighbours are (clamped at the walls, where
    // the coefficient is 0.0; the z neighbours of the slab's end planes in the neighbour CTA).
    const int hx = (g.nx + 1) >> 1;
    const int items = hx * g.ny * pz;
    int n0[CL_ITEMS], m0[CL_ITEMS], par[CL_ITEMS], edge[CL_ITEMS];
#pragma unroll
    for (int q = 0; q < CL_ITEMS; ++q) {
        const int h = (int)threadIdx.x + q * CL_THREADS;
        n0[q] = -1;
        m0[q] = par[q] = edge[q] = 0;
        if (h < items) {
            const int ih = h % hx, t = h / hx;
            const int j = t % g.ny, kl = t / g.ny;
            m0[q] = 2 * ih + g.nx * j;                            // index inside a plane
            n0[q] = m0[q] + plane * kl;
            par[q] = (j + k0 + kl) & 1;                           // the red cell of the pair: i = 2 ih + par
            edge[q] = (2 * ih == 0 ? 1 : 0) | (2 * ih + 2 >= g.nx ? 2 : 0) | (j == 0 ? 4 : 0) |
                      (j == g.ny - 1 ? 8 : 0) | (kl == 0 ? 16 : 0) | (kl == pz - 1 ? 32 : 0) |
                      (2 * ih + 1 >= g.nx ? 64 : 0);              // odd nx: the pair has one cell
        }
    }
    for (int s = 0; s < 2 * nsweeps; ++s) {
        const int colour = s & 1;
#pragma unroll
        for (int q = 0; q < CL_ITEMS; ++q) {
            if (n0[q] < 0) continue;
            const int off = par[q] ^ colour;                      // 0: left cell, 1: right cell
            const int e = edge[q];
            if (off && (e & 64)) continue;
            const int n = n0[q] + off;
            const bool wxm = (e & 1) && !off, wxp = (e & 2) && (off || (e & 64));
            const int m = m0[q] + off;
            const double axm = wxm ? 0.0 : AX[n - 1], axp = AX[n];
            const double aym = (e & 4) ? 0.0 : AY[n - g.nx], ayp = AY[n];
            const double azm = AZ[n], azp = AZ[n + plane];
            const double pxm = P[wxm ? n : n - 1];
            const double pxp = P[wxp ? n : n + 1];
            const double pym = P[(e & 4) ? n : n - g.nx];
            const double pyp = P[(e & 8) ? n : n + g.nx];
            const double pzm = (e & 16) ? Pdn[(pz - 1) * plane + m] : P[n - plane];
            const double pzp = (e & 32) ? Pup[m] : P[n + plane];
            P[n] = sor_update(axm, axp, aym, ayp, azm, azp, pxm, pxp, pym, pyp, pzm, pzp, P[n],
                              RH[n], omega);
        }
        cluster.sync();      // the colour just written is read by everybody in the next half-sweep
    }
    for (int n = threadIdx.x; n < slab; n += CL_THREADS) p[base + n] = P[n];
}

// One-time set-up of the kernel's attributes; returns the cluster size this device can run for
// the grid (0: not available).
inline int cl_plan(const Grid &g)
{
    const int C = cl_cluster_size(g);
    if (C == 0) return 0;
    if (cudaFuncSetAttribute(ps_cluster_sweeps_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)CL_SMEM_MAX) != cudaSuccess ||
        cudaFuncSetAttribute(ps_cluster_sweeps_kernel,
                             cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)C);
    cfg.blockDim = dim3(CL_THREADS);
    cfg.dynamicSmemBytes = cl_smem_bytes(g, C);
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, ps_cluster_sweeps_kernel, &cfg) != cudaSuccess ||
        nclusters < 1) {
        cudaGetLastError();
        return 0;
    }
    return C;
}

inline cudaError_t cl_launch(const Grid &g, int C, const double *ax, const double *ay,
                             const double *az, const double *rhs, double *p, double omega,
                             int nsweeps, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)C);
    cfg.blockDim = dim3(CL_THREADS);
    cfg.dynamicSmemBytes = cl_smem_bytes(g, C);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, ps_cluster_sweeps_kernel, g, ax, ay, az, rhs, p, omega, nsweeps);
}

}  // namespace ps
