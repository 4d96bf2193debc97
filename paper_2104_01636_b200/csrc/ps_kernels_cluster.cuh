// ps_kernels_cluster.cuh -- many red-black SOR sweeps in ONE launch for grids that fit the shared
// memory of one thread-block cluster (sm_100a: up to 16 CTAs x 227 KB).
//
// The smallest grids (BASELINE.json config 1; the coarse levels of the multigrid hierarchy, which
// run 48 sweeps per visit) are bound by synchronisation latency, not by bandwidth: the resident
// kernel (ps_kernels_resident.cuh) spends 2.6 us per half-sweep on a grid-wide barrier through
// global memory and on L2 round trips.  Here the whole problem lives on chip for the launch:
//   * the launch is ONE cluster of C CTAs (C = 16, 8, 4, 2 or 1, the largest that divides nz);
//     CTA r owns the z slab [r nz/C, (r+1) nz/C) and keeps p, ax, ay, rhs of the slab and az of
//     the slab plus the plane below it in shared memory (loaded once, p written back once),
//     each field colour-compacted (see cl_smem_bytes);
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

// Shared memory of one CTA.  Every field is stored COLOUR-COMPACTED: one array per colour, entry
// ih + hx (j + ny kl) with hx = ceil(nx / 2) holding the cell of that colour in the x-pair ih of row
// (j, kl).  A half-sweep then reads its own colour's entry and the other colour's neighbours at
// unit stride across a warp (2 shared-memory wavefronts per 8-byte access instead of the 4 of a
// natural layout read at stride 2, which made the shared-memory pipe the limit at 65 k cells).
// 4 slab fields (p, ax, ay, rhs) + az with one extra plane below the slab, two colours each.
inline size_t cl_smem_bytes(const Grid &g, int C)
{
    const size_t planec = (size_t)((g.nx + 1) / 2) * g.ny, pz = (size_t)(g.nz / C);
    return 2 * (4 * pz * planec + (pz + 1) * planec) * sizeof(double);
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
    const int hx = (g.nx + 1) >> 1;
    const int plane = g.nx * g.ny, slab = pz * plane;       // natural layout (global memory)
    const int planec = hx * g.ny, slabc = pz * planec;      // one colour (shared memory)
    // per colour c: P[c], AX[c], AY[c], RH[c] of slabc entries; AZ[c] of slabc + planec entries,
    // its first plane = az of the plane below the slab (periodic)
    // (addresses by arithmetic: arrays of pointers indexed by the colour would live in local memory)
    auto fP = [&](int c) { return cl_smem + c * slabc; };
    auto fAX = [&](int c) { return cl_smem + (2 + c) * slabc; };
    auto fAY = [&](int c) { return cl_smem + (4 + c) * slabc; };
    auto fRH = [&](int c) { return cl_smem + (6 + c) * slabc; };
    auto fAZ = [&](int c) { return cl_smem + 8 * slabc + c * (slabc + planec); };
    const size_t base = (size_t)k0 * plane;
    for (int n = threadIdx.x; n < slab; n += CL_THREADS) {
        const int i = n % g.nx, t = n / g.nx;
        const int j = t % g.ny, kl = t / g.ny;
        const int c = (i + j + k0 + kl) & 1, q = (i >> 1) + hx * (j + g.ny * kl);
        fP(c)[q] = p[base + n];
        fAX(c)[q] = ax[base + n];
        fAY(c)[q] = ay[base + n];
        fRH(c)[q] = rhs[base + n];
        fAZ(c)[planec + q] = az[base + n];
    }
    const size_t below = (size_t)(k0 > 0 ? k0 - 1 : g.nz - 1) * plane;
    for (int n = threadIdx.x; n < plane; n += CL_THREADS) {
        const int i = n % g.nx, j = n / g.nx;
        fAZ((i + j + k0 + 1) & 1)[(i >> 1) + hx * j] = az[below + n];     // plane k0 - 1
    }
    // the slabs of the z neighbours (the CTA itself when the cluster is one CTA: periodic)
    const int rdn = rank > 0 ? rank - 1 : C - 1, rup = rank + 1 < C ? rank + 1 : 0;
    const double *Pdn0 = cluster.map_shared_rank(cl_smem, rdn);       // their P of colour 0
    const double *Pup0 = cluster.map_shared_rank(cl_smem, rup);
    cluster.sync();

    // A thread keeps the same (at most CL_ITEMS) x-pairs of cells for the whole launch -- in each
    // half-sweep it updates the cell of the pair that has the active colour -- so everything that
    // does not depend on the colour is worked out once, here.
    const int items = slabc;
    int m0[CL_ITEMS], par[CL_ITEMS], edge[CL_ITEMS];
#pragma unroll
    for (int q = 0; q < CL_ITEMS; ++q) {
        const int h = (int)threadIdx.x + q * CL_THREADS;
        m0[q] = -1;
        par[q] = edge[q] = 0;
        if (h < items) {
            const int ih = h % hx, t = h / hx;
            const int j = t % g.ny, kl = t / g.ny;
            m0[q] = ih + hx * j;                                  // entry inside a plane
            par[q] = (j + k0 + kl) & 1;                           // the pair's red cell: i = 2 ih + par
            edge[q] = (ih == 0 ? 1 : 0) | (2 * ih == g.nx - 1 ? 2 : 0) | (2 * ih + 1 == g.nx - 1 ? 128 : 0) |
                      (j == 0 ? 4 : 0) | (j == g.ny - 1 ? 8 : 0) | (kl == 0 ? 16 : 0) |
                      (kl == pz - 1 ? 32 : 0) | (2 * ih + 1 >= g.nx ? 64 : 0);   // 64: odd nx, one cell
        }
    }
    for (int s = 0; s < 2 * nsweeps; ++s) {
        const int c = s & 1, o = c ^ 1;                           // active colour, the other colour
        double *Pc = fP(c);
        const double *Po = fP(o), *AXc = fAX(c), *AXo = fAX(o), *AYc = fAY(c), *AYo = fAY(o),
                     *AZc = fAZ(c), *AZo = fAZ(o), *RHc = fRH(c);
        const double *Pdn = Pdn0 + o * slabc, *Pup = Pup0 + o * slabc;
#pragma unroll
        for (int q = 0; q < CL_ITEMS; ++q) {
            if (m0[q] < 0) continue;
            const int off = par[q] ^ c;                           // 0: left cell of the pair, 1: right
            const int e = edge[q];
            if (off && (e & 64)) continue;
            const int n = (int)threadIdx.x + q * CL_THREADS;      // entry in the colour arrays
            const bool wxm = (e & 1) && !off;                     // the cell is at the x- / x+ wall
            const bool wxp = off ? (e & 128) != 0 : (e & 2) != 0;
            const double pc = Pc[n];
            const double axm = wxm ? 0.0 : AXo[n - 1 + off], axp = AXc[n];
            const double aym = (e & 4) ? 0.0 : AYo[n - hx], ayp = AYc[n];
            const double azm = AZo[n], azp = AZc[n + planec];
            const double pxm = wxm ? pc : Po[n - 1 + off];
            const double pxp = wxp ? pc : Po[n + off];
            const double pym = (e & 4) ? pc : Po[n - hx];
            const double pyp = (e & 8) ? pc : Po[n + hx];
            const double pzm = (e & 16) ? Pdn[(pz - 1) * planec + m0[q]] : Po[n - planec];
            const double pzp = (e & 32) ? Pup[m0[q]] : Po[n + planec];
            Pc[n] = sor_update(axm, axp, aym, ayp, azm, azp, pxm, pxp, pym, pyp, pzm, pzp, pc,
                               RHc[n], omega);
        }
        cluster.sync();      // the colour just written is read by everybody in the next half-sweep
    }
    for (int n = threadIdx.x; n < slab; n += CL_THREADS) {
        const int i = n % g.nx, t = n / g.nx;
        const int j = t % g.ny, kl = t / g.ny;
        p[base + n] = fP((i + j + k0 + kl) & 1)[(i >> 1) + hx * (j + g.ny * kl)];
    }
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
    cudaLaunchConfig_t cfg = {};
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
    cudaLaunchConfig_t cfg = {};
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
