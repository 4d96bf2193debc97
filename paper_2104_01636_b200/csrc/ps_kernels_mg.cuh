// ps_kernels_mg.cuh -- grid-transfer kernels of the multigrid acceleration (PAPER.md:78
// "multigrid accelerated red black SOR relaxation scheme"; readings M1-M4 of DESIGN.md §12).
//
//   ps_mg_coarsen_kernel          M1  coarse face coefficient = 1/16 sum of the 4 fine faces
//   ps_mg_residual_restrict_pair_kernel M2+M3  rc = 1/8 sum over the 8 children of (rhs - A p)
//   ps_mg_prolong_add_kernel      M4  p += e_parent
//
// All are single-pass, HBM-bound streaming kernels: one thread per COARSE cell (coarsen,
// residual+restrict: it reads its 2x2x2 children with 16-byte loads) or per pair of fine cells
// (prolongation).  The summation orders are fixed and written out, so results are bitwise those
// of the two-step definition (residual field, then restriction).  Compile with --fmad=false.
#pragma once
#include "ps_kernels_generic.cuh"

namespace ps {

// M1.  gf = fine grid (nx, ny even; nz even).  Coarse cell (I,J,K); fine corner (2I,2J,2K).
__global__ void __launch_bounds__(256)
ps_mg_coarsen_kernel(Grid gf, const double *__restrict__ ax, const double *__restrict__ ay,
                     const double *__restrict__ az, double *__restrict__ axc,
                     double *__restrict__ ayc, double *__restrict__ azc)
{
    const int cx = gf.nx >> 1, cy = gf.ny >> 1, cz = gf.nz >> 1;
    const size_t NC = (size_t)cx * cy * cz;
    const size_t sx = 1, sy = (size_t)gf.nx, sz = (size_t)gf.nx * gf.ny;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < NC;
         c += (size_t)gridDim.x * blockDim.x) {
        const int I = (int)((unsigned)c % (unsigned)cx);
        const unsigned t = (unsigned)c / (unsigned)cx;
        const int J = (int)(t % (unsigned)cy), K = (int)(t / (unsigned)cy);
        const size_t n = gf.idx(2 * I, 2 * J, 2 * K);
        axc[c] = 0.0625 * (((ax[n + sx] + ax[n + sx + sy]) + ax[n + sx + sz]) + ax[n + sx + sy + sz]);
        ayc[c] = 0.0625 * (((ay[n + sy] + ay[n + sx + sy]) + ay[n + sy + sz]) + ay[n + sx + sy + sz]);
        azc[c] = 0.0625 * (((az[n + sz] + az[n + sx + sz]) + az[n + sy + sz]) + az[n + sx + sy + sz]);
    }
}

// M2 + M3 fused: the residual of the 8 children (4 x-pairs, 16-byte loads), summed with x fastest,
// then y, then z, times 1/8.  The residual field itself is never stored (saves 16 B per fine cell
// of traffic).  nx is even on every level that is coarsened.
__global__ void __launch_bounds__(256)
ps_mg_residual_restrict_pair_kernel(Grid gf, const double *__restrict__ ax,
                                    const double *__restrict__ ay, const double *__restrict__ az,
                                    const double *__restrict__ rhs, const double *__restrict__ p,
                                    double *__restrict__ rc)
{
    const int cx = gf.nx >> 1, cy = gf.ny >> 1, cz = gf.nz >> 1;
    const size_t NC = (size_t)cx * cy * cz;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < NC;
         c += (size_t)gridDim.x * blockDim.x) {
        const int I = (int)((unsigned)c % (unsigned)cx);
        const unsigned t = (unsigned)c / (unsigned)cx;
        const int J = (int)(t % (unsigned)cy), K = (int)(t / (unsigned)cy);
        double acc = 0.0;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = 2 * I, j = 2 * J + (q & 1), k = 2 * K + (q >> 1);
            double2 b;
            const double2 r = residual_pair(gf, ax, ay, az, rhs, p, i, j, k, gf.idx(i, j, k), b);
            acc = (q == 0) ? r.x : acc + r.x;
            acc = acc + r.y;
        }
        rc[c] = 0.125 * acc;
    }
}

// M2 + M3 + the norms of row a4 in one pass (used by ps_mg_solve when the finest level has no
// pre-smoothing: the residual the restriction needs is then the residual of the iterate whose
// norm decides the stop, so the separate 40 B/cell norm pass of every cycle is saved).
// Block b owns the coarse cells [512 b, 512 b + 512) = RED_CHUNK fine cells; thread t takes
// coarse cells t and t + 256 of them and adds r^2 (and rhs^2) of its 16 children in the order
// (x, y, z fastest to slowest), then the fixed block tree: the partials depend on N only, like
// those of ps_residual_partial_kernel (a different, equally fixed tree: the two norms agree to
// rounding, not bitwise).
__global__ void __launch_bounds__(RED_THREADS)
ps_mg_residual_restrict_norm_kernel(Grid gf, const double *__restrict__ ax,
                                    const double *__restrict__ ay, const double *__restrict__ az,
                                    const double *__restrict__ rhs, const double *__restrict__ p,
                                    double *__restrict__ rc, double *__restrict__ partR2,
                                    double *__restrict__ partB2)
{
    __shared__ double sm[RED_THREADS / 32];
    const int cx = gf.nx >> 1, cy = gf.ny >> 1, cz = gf.nz >> 1;
    const size_t NC = (size_t)cx * cy * cz;
    const size_t base = (size_t)blockIdx.x * (RED_CHUNK / 8);
    double r2 = 0.0, b2 = 0.0;
#pragma unroll 1
    for (int m = 0; m < RED_CHUNK / 8 / RED_THREADS; ++m) {
        const size_t c = base + (size_t)m * RED_THREADS + threadIdx.x;
        if (c < NC) {
            const int I = (int)((unsigned)c % (unsigned)cx);
            const unsigned t = (unsigned)c / (unsigned)cx;
            const int J = (int)(t % (unsigned)cy), K = (int)(t / (unsigned)cy);
            double acc = 0.0;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = 2 * I, j = 2 * J + (q & 1), k = 2 * K + (q >> 1);
                double2 b;
                const double2 r = residual_pair(gf, ax, ay, az, rhs, p, i, j, k, gf.idx(i, j, k), b);
                acc = (q == 0) ? r.x : acc + r.x;
                acc = acc + r.y;
                r2 = r2 + r.x * r.x;
                r2 = r2 + r.y * r.y;
                b2 = b2 + b.x * b.x;
                b2 = b2 + b.y * b.y;
            }
            rc[c] = 0.125 * acc;
        }
    }
    const double Rs = block_tree_sum<RED_THREADS>(r2, sm);
    const double Bs = block_tree_sum<RED_THREADS>(b2, sm);
    if (threadIdx.x == 0) {
        partR2[blockIdx.x] = Rs;
        partB2[blockIdx.x] = Bs;
    }
}

// M4.  One thread per x-pair of fine cells (both children of the same parent): 16-byte access.
__global__ void __launch_bounds__(256)
ps_mg_prolong_add_kernel(Grid gf, const double *__restrict__ ec, double *__restrict__ p)
{
    const int cx = gf.nx >> 1, cy = gf.ny >> 1;
    const size_t pairs = (size_t)cx * gf.ny * gf.nz;
    for (size_t h = (size_t)blockIdx.x * blockDim.x + threadIdx.x; h < pairs;
         h += (size_t)gridDim.x * blockDim.x) {
        const int I = (int)((unsigned)h % (unsigned)cx);
        const unsigned t = (unsigned)h / (unsigned)cx;
        const int j = (int)(t % (unsigned)gf.ny), k = (int)(t / (unsigned)gf.ny);
        const double e = ec[(size_t)I + (size_t)cx * ((size_t)(j >> 1) + (size_t)cy * (size_t)(k >> 1))];
        double2 *q = reinterpret_cast<double2 *>(p + gf.idx(2 * I, j, k));
        double2 v = *q;
        v.x = v.x + e;
        v.y = v.y + e;
        *q = v;
    }
}

}  // namespace ps
