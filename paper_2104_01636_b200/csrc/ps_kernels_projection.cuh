// ps_kernels_projection.cuh -- the steps either side of the pressure solve (PAPER.md:107-115,
// steps 10-12 of the time step; readings P1-P3 of DESIGN.md §13):
//
//   ps_rhs_from_velocity_kernel   rhs = div(u^_f)/dt, u^_f = linear average c->f (0 on walls)
//   ps_correct_velocity_kernel    u_c <- u^_c - dt (grad p/rho)_{f->c}
//   ps_face_divergence_kernel     div(u^_f - dt (grad p/rho)_f)   (= dt (rhs - A p))
//
// Single-pass streaming kernels, one thread per cell, natural layout, neighbour reuse through
// L1/L2; HBM-bound: 32 B/cell (rhs), 80 B/cell (correction: p 8, coefficients 24, u 24 + 24),
// 64 B/cell (face divergence).  Expression order = the oracle's (compile with --fmad=false).
#pragma once
#include "ps_kernels_generic.cuh"

namespace ps {

struct Spacing { double dx, dy, dz; };

__device__ __forceinline__ void cell_of(const Grid &g, size_t n, int &i, int &j, int &k)
{
    i = (int)((unsigned)n % (unsigned)g.nx);
    const unsigned t = (unsigned)n / (unsigned)g.nx;
    j = (int)(t % (unsigned)g.ny);
    k = (int)(t / (unsigned)g.ny);
}

// f[0..5] = x-, x+, y-, y+, z-, z+ face-normal velocities of cell n.
__device__ __forceinline__ void face_velocities(const Grid &g, const double *__restrict__ ux,
                                                const double *__restrict__ uy,
                                                const double *__restrict__ uz, int i, int j, int k,
                                                size_t n, double f[6])
{
    const size_t plane = (size_t)g.nx * g.ny;
    const size_t nzm = (k > 0) ? n - plane : n + plane * (size_t)(g.nz - 1);
    const size_t nzp = (k + 1 < g.nz) ? n + plane : n - plane * (size_t)(g.nz - 1);
    const double uxc = ux[n], uyc = uy[n], uzc = uz[n];
    f[0] = (i > 0) ? 0.5 * (ux[n - 1] + uxc) : 0.0;
    f[1] = (i < g.nx - 1) ? 0.5 * (uxc + ux[n + 1]) : 0.0;
    f[2] = (j > 0) ? 0.5 * (uy[n - g.nx] + uyc) : 0.0;
    f[3] = (j < g.ny - 1) ? 0.5 * (uyc + uy[n + g.nx]) : 0.0;
    f[4] = 0.5 * (uz[nzm] + uzc);
    f[5] = 0.5 * (uzc + uz[nzp]);
}

// g6[0..5] = (grad p / rho) . n on the same faces: a_f h (p_nb - p_c), 0 on walls.
__device__ __forceinline__ void face_gradients(const Grid &g, const Spacing &h,
                                               const double *__restrict__ ax,
                                               const double *__restrict__ ay,
                                               const double *__restrict__ az,
                                               const double *__restrict__ p, int i, int j, int k,
                                               size_t n, double g6[6])
{
    const Stencil s = gather(g, ax, ay, az, p, i, j, k, n);
    const double pc = p[n];
    g6[0] = (s.axm * h.dx) * (pc - s.pxm);
    g6[1] = (s.axp * h.dx) * (s.pxp - pc);
    g6[2] = (s.aym * h.dy) * (pc - s.pym);
    g6[3] = (s.ayp * h.dy) * (s.pyp - pc);
    g6[4] = (s.azm * h.dz) * (pc - s.pzm);
    g6[5] = (s.azp * h.dz) * (s.pzp - pc);
}

__global__ void __launch_bounds__(256)
ps_rhs_from_velocity_kernel(Grid g, Spacing h, const double *__restrict__ ux,
                            const double *__restrict__ uy, const double *__restrict__ uz,
                            double dt, double *__restrict__ rhs)
{
    const size_t N = g.cells();
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < N;
         n += (size_t)gridDim.x * blockDim.x) {
        int i, j, k;
        cell_of(g, n, i, j, k);
        double f[6];
        face_velocities(g, ux, uy, uz, i, j, k, n, f);
        const double div = (((f[1] - f[0]) / h.dx) + ((f[3] - f[2]) / h.dy)) + ((f[5] - f[4]) / h.dz);
        rhs[n] = div / dt;
    }
}

// In place on u: a cell only reads p and the coefficients of its neighbours, never their u.
__global__ void __launch_bounds__(256)
ps_correct_velocity_kernel(Grid g, Spacing h, const double *__restrict__ ax,
                           const double *__restrict__ ay, const double *__restrict__ az,
                           const double *__restrict__ p, double dt, double *ux, double *uy,
                           double *uz)
{
    const size_t N = g.cells();
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < N;
         n += (size_t)gridDim.x * blockDim.x) {
        int i, j, k;
        cell_of(g, n, i, j, k);
        double q[6];
        face_gradients(g, h, ax, ay, az, p, i, j, k, n, q);
        ux[n] = ux[n] - dt * (0.5 * (q[0] + q[1]));
        uy[n] = uy[n] - dt * (0.5 * (q[2] + q[3]));
        uz[n] = uz[n] - dt * (0.5 * (q[4] + q[5]));
    }
}

__global__ void __launch_bounds__(256)
ps_face_divergence_kernel(Grid g, Spacing h, const double *__restrict__ ax,
                          const double *__restrict__ ay, const double *__restrict__ az,
                          const double *__restrict__ ux, const double *__restrict__ uy,
                          const double *__restrict__ uz, const double *__restrict__ p, double dt,
                          double *__restrict__ div)
{
    const size_t N = g.cells();
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < N;
         n += (size_t)gridDim.x * blockDim.x) {
        int i, j, k;
        cell_of(g, n, i, j, k);
        double f[6], q[6], u[6];
        face_velocities(g, ux, uy, uz, i, j, k, n, f);
        face_gradients(g, h, ax, ay, az, p, i, j, k, n, q);
#pragma unroll
        for (int m = 0; m < 6; ++m) u[m] = f[m] - dt * q[m];
        div[n] = (((u[1] - u[0]) / h.dx) + ((u[3] - u[2]) / h.dy)) + ((u[5] - u[4]) / h.dz);
    }
}

}  // namespace ps

// ---------------------------------------------------------------------------------------------
// Sharp-surface-force right-hand side of the p~ system (eqs (6)-(7)):
//   rhs_c = - sum_f a_f (sigma kappa_f) (F_nb - F_c),  kappa_f = 0.5 (kappa_c + kappa_nb).
// One thread per cell; F 8 + kappa 8 + coefficients 24 read, 8 written = 48 B/cell.
namespace ps {

__global__ void __launch_bounds__(256)
ps_ssf_rhs_kernel(Grid g, const double *__restrict__ ax, const double *__restrict__ ay,
                  const double *__restrict__ az, const double *__restrict__ F,
                  const double *__restrict__ kappa, double sigma, double *__restrict__ rhs)
{
    const size_t N = g.cells();
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < N;
         n += (size_t)gridDim.x * blockDim.x) {
        int i, j, k;
        cell_of(g, n, i, j, k);
        const size_t plane = (size_t)g.nx * g.ny;
        const size_t nzm = (k > 0) ? n - plane : n + plane * (size_t)(g.nz - 1);
        const size_t nzp = (k + 1 < g.nz) ? n + plane : n - plane * (size_t)(g.nz - 1);
        const size_t nb[6] = {(i > 0) ? n - 1 : n, (i < g.nx - 1) ? n + 1 : n,
                              (j > 0) ? n - g.nx : n, (j < g.ny - 1) ? n + g.nx : n, nzm, nzp};
        const double a[6] = {(i > 0) ? ax[n - 1] : 0.0, ax[n], (j > 0) ? ay[n - g.nx] : 0.0, ay[n],
                             az[nzm], az[n]};
        const double Fc = F[n], kc = kappa[n];
        double t[6];
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            const double kf = 0.5 * (kc + kappa[nb[q]]);
            t[q] = (a[q] * (sigma * kf)) * (F[nb[q]] - Fc);
        }
        rhs[n] = -(((((t[0] + t[1]) + t[2]) + t[3]) + t[4]) + t[5]);
    }
}

}  // namespace ps
