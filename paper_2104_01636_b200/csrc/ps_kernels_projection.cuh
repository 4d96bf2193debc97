// ps_kernels_projection.cuh -- the steps either side of the pressure solve (PAPER.md:107-115,
// steps 10-12 of the time step; readings P1-P3 of DESIGN.md §13):
//
//   ps_rhs_from_velocity_kernel   rhs = div(u^_f)/dt, u^_f = linear average c->f (0 on walls)
//   ps_correct_velocity_kernel    u_c <- u^_c - dt (grad p/rho)_{f->c}
//   ps_face_divergence_kernel     div(u^_f - dt (grad p/rho)_f)   (= dt (rhs - A p))
//
// single-pass streaming kernels, one thread per cell (per x-pair of cells for even nx), natural layout, neighbour reuse through
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

// ---------------------------------------------------------------------------------------------
// The same three-field stencils for even nx and 16-byte aligned arrays: one thread per x-pair of
// cells (n, n+1), 16-byte loads and stores, 32-bit pair index.  Every value is produced by the
// same expression as in the one-cell kernels above.
struct PairCell { int i, j, k; size_t n, nzm, nzp; };

__device__ __forceinline__ PairCell pair_cell(const Grid &g, unsigned h)
{
    const unsigned hx = (unsigned)g.nx >> 1;
    PairCell c;
    c.i = 2 * (int)(h % hx);
    const unsigned t = h / hx;
    c.j = (int)(t % (unsigned)g.ny);
    c.k = (int)(t / (unsigned)g.ny);
    c.n = g.idx(c.i, c.j, c.k);
    const size_t plane = (size_t)g.nx * g.ny;
    c.nzm = (c.k > 0) ? c.n - plane : c.n + plane * (size_t)(g.nz - 1);
    c.nzp = (c.k + 1 < g.nz) ? c.n + plane : c.n - plane * (size_t)(g.nz - 1);
    return c;
}

// z-marching form of the pair stencils.  A block is a tile of 32 x-pairs (64 cells) x 8 rows, a
// thread owns one x-pair and marches it through a chunk of z planes, carrying what the stencil
// needs of the planes k-1, k, k+1 (uz; p and az for the face divergence) in registers: every
// plane of those fields is loaded once per chunk instead of three times.  Read through L1/L2 like
// the one-cell kernels, the z neighbours alone were 1/3 of the load instructions and of the L2
// traffic, and the kernels ran at 0.8 of the HBM roofline, bound by L2 bandwidth.
constexpr int ZS_TX = 32, ZS_TY = 8;

struct ZsCell { int i, j; size_t n; };     // left cell of the pair and its linear index on plane k

// fa[0..5], fb[0..5]: face velocities of the left and the right cell of the pair; UZm, UZ, UZp:
// the uz pair on planes k-1, k, k+1.
__device__ __forceinline__ void face_velocities_pair(const Grid &g, const double *__restrict__ ux,
                                                     const double *__restrict__ uy,
                                                     const ZsCell &c, const double2 UZm,
                                                     const double2 UZ, const double2 UZp,
                                                     double fa[6], double fb[6])
{
    const double2 UX = ld2(ux + c.n), UY = ld2(uy + c.n);
    const double mid = 0.5 * (UX.x + UX.y);
    fa[0] = (c.i > 0) ? 0.5 * (ux[c.n - 1] + UX.x) : 0.0;
    fa[1] = mid;
    fb[0] = mid;
    fb[1] = (c.i + 2 < g.nx) ? 0.5 * (UX.y + ux[c.n + 2]) : 0.0;
    fa[2] = fb[2] = fa[3] = fb[3] = 0.0;
    if (c.j > 0) {
        const double2 U = ld2(uy + c.n - g.nx);
        fa[2] = 0.5 * (U.x + UY.x);
        fb[2] = 0.5 * (U.y + UY.y);
    }
    if (c.j < g.ny - 1) {
        const double2 U = ld2(uy + c.n + g.nx);
        fa[3] = 0.5 * (UY.x + U.x);
        fb[3] = 0.5 * (UY.y + U.y);
    }
    fa[4] = 0.5 * (UZm.x + UZ.x);
    fb[4] = 0.5 * (UZm.y + UZ.y);
    fa[5] = 0.5 * (UZ.x + UZp.x);
    fb[5] = 0.5 * (UZ.y + UZp.y);
}

// ga[0..5], gb[0..5]: (grad p / rho) . n on the faces of the two cells (face_gradients per cell);
// Pzm, P, Pzp: the p pair on planes k-1, k, k+1; AZm, AZ: the az pair on planes k-1, k.
__device__ __forceinline__ void face_gradients_pair(const Grid &g, const Spacing &h,
                                                    const double *__restrict__ ax,
                                                    const double *__restrict__ ay,
                                                    const double *__restrict__ p, const ZsCell &c,
                                                    const double2 AZm, const double2 AZ,
                                                    const double2 Pzm, const double2 P,
                                                    const double2 Pzp, double ga[6], double gb[6])
{
    const double2 AX = ld2(ax + c.n), AY = ld2(ay + c.n);
    const double axl = (c.i > 0) ? ax[c.n - 1] : 0.0;
    const double pl = p[(c.i > 0) ? c.n - 1 : c.n];
    const double pr = p[(c.i + 2 < g.nx) ? c.n + 2 : c.n + 1];
    const double2 AYm = (c.j > 0) ? ld2(ay + c.n - g.nx) : make_double2(0.0, 0.0);
    const double2 Pym = ld2(p + ((c.j > 0) ? c.n - g.nx : c.n));
    const double2 Pyp = ld2(p + ((c.j < g.ny - 1) ? c.n + g.nx : c.n));
    ga[0] = (axl * h.dx) * (P.x - pl);
    ga[1] = (AX.x * h.dx) * (P.y - P.x);
    gb[0] = (AX.x * h.dx) * (P.y - P.x);
    gb[1] = (AX.y * h.dx) * (pr - P.y);
    ga[2] = (AYm.x * h.dy) * (P.x - Pym.x);
    gb[2] = (AYm.y * h.dy) * (P.y - Pym.y);
    ga[3] = (AY.x * h.dy) * (Pyp.x - P.x);
    gb[3] = (AY.y * h.dy) * (Pyp.y - P.y);
    ga[4] = (AZm.x * h.dz) * (P.x - Pzm.x);
    gb[4] = (AZm.y * h.dz) * (P.y - Pzm.y);
    ga[5] = (AZ.x * h.dz) * (Pzp.x - P.x);
    gb[5] = (AZ.y * h.dz) * (Pzp.y - P.y);
}

// Grid of the z-marching kernels: x tiles, y tiles, z chunks of kz planes.
__device__ __forceinline__ bool zs_setup(const Grid &g, int kz, ZsCell &c, int &k0, int &k1,
                                         size_t &plane, size_t &nzm)
{
    c.i = 2 * ((int)blockIdx.x * ZS_TX + (int)(threadIdx.x & 31u));
    c.j = (int)blockIdx.y * ZS_TY + (int)(threadIdx.x >> 5);
    k0 = (int)blockIdx.z * kz;
    k1 = k0 + kz < g.nz ? k0 + kz : g.nz;
    if (c.i >= g.nx || c.j >= g.ny || k0 >= k1) return false;
    plane = (size_t)g.nx * g.ny;
    c.n = g.idx(c.i, c.j, k0);
    nzm = (k0 > 0) ? c.n - plane : c.n + plane * (size_t)(g.nz - 1);
    return true;
}

__global__ void __launch_bounds__(ZS_TX * ZS_TY)
ps_rhs_from_velocity_pair_kernel(Grid g, Spacing h, const double *__restrict__ ux,
                                 const double *__restrict__ uy, const double *__restrict__ uz,
                                 double dt, double *__restrict__ rhs, int kz)
{
    ZsCell c;
    int k0, k1;
    size_t plane, nzm;
    if (!zs_setup(g, kz, c, k0, k1, plane, nzm)) return;
    double2 UZm = ld2(uz + nzm), UZ = ld2(uz + c.n);
    for (int k = k0; k < k1; ++k, c.n += plane) {
        const size_t nzp = (k + 1 < g.nz) ? c.n + plane : c.n - plane * (size_t)(g.nz - 1);
        const double2 UZp = ld2(uz + nzp);
        double fa[6], fb[6];
        face_velocities_pair(g, ux, uy, c, UZm, UZ, UZp, fa, fb);
        const double da = (((fa[1] - fa[0]) / h.dx) + ((fa[3] - fa[2]) / h.dy)) + ((fa[5] - fa[4]) / h.dz);
        const double db = (((fb[1] - fb[0]) / h.dx) + ((fb[3] - fb[2]) / h.dy)) + ((fb[5] - fb[4]) / h.dz);
        *reinterpret_cast<double2 *>(rhs + c.n) = make_double2(da / dt, db / dt);
        UZm = UZ;
        UZ = UZp;
    }
}

__global__ void __launch_bounds__(ZS_TX * ZS_TY, 3)
ps_face_divergence_pair_kernel(Grid g, Spacing h, const double *__restrict__ ax,
                               const double *__restrict__ ay, const double *__restrict__ az,
                               const double *__restrict__ ux, const double *__restrict__ uy,
                               const double *__restrict__ uz, const double *__restrict__ p,
                               double dt, double *__restrict__ div, int kz)
{
    ZsCell c;
    int k0, k1;
    size_t plane, nzm;
    if (!zs_setup(g, kz, c, k0, k1, plane, nzm)) return;
    double2 UZm = ld2(uz + nzm), UZ = ld2(uz + c.n);
    double2 Pzm = ld2(p + nzm), P = ld2(p + c.n);
    double2 AZm = ld2(az + nzm);
    for (int k = k0; k < k1; ++k, c.n += plane) {
        const size_t nzp = (k + 1 < g.nz) ? c.n + plane : c.n - plane * (size_t)(g.nz - 1);
        const double2 UZp = ld2(uz + nzp), Pzp = ld2(p + nzp), AZ = ld2(az + c.n);
        double fa[6], fb[6], ga[6], gb[6], ua[6], ub[6];
        face_velocities_pair(g, ux, uy, c, UZm, UZ, UZp, fa, fb);
        face_gradients_pair(g, h, ax, ay, p, c, AZm, AZ, Pzm, P, Pzp, ga, gb);
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            ua[m] = fa[m] - dt * ga[m];
            ub[m] = fb[m] - dt * gb[m];
        }
        const double da = (((ua[1] - ua[0]) / h.dx) + ((ua[3] - ua[2]) / h.dy)) + ((ua[5] - ua[4]) / h.dz);
        const double db = (((ub[1] - ub[0]) / h.dx) + ((ub[3] - ub[2]) / h.dy)) + ((ub[5] - ub[4]) / h.dz);
        *reinterpret_cast<double2 *>(div + c.n) = make_double2(da, db);
        UZm = UZ; UZ = UZp;
        Pzm = P; P = Pzp;
        AZm = AZ;
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

// One thread per x-pair (even nx, 16-byte aligned arrays); the same expressions per cell.
__device__ __forceinline__ double ssf_term(double a, double sigma, double kc, double kn, double Fc,
                                           double Fn)
{
    const double kf = 0.5 * (kc + kn);
    return (a * (sigma * kf)) * (Fn - Fc);
}

__global__ void __launch_bounds__(256)
ps_ssf_rhs_pair_kernel(Grid g, const double *__restrict__ ax, const double *__restrict__ ay,
                       const double *__restrict__ az, const double *__restrict__ F,
                       const double *__restrict__ kappa, double sigma, double *__restrict__ rhs)
{
    const unsigned pairs = ((unsigned)g.nx >> 1) * (unsigned)g.ny * (unsigned)g.nz;
    for (unsigned q = blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += gridDim.x * blockDim.x) {
        const PairCell c = pair_cell(g, q);
        const size_t n = c.n;
        const double2 Fc = ld2(F + n), Kc = ld2(kappa + n);
        const double2 AX = ld2(ax + n), AY = ld2(ay + n), AZ = ld2(az + n), AZm = ld2(az + c.nzm);
        const double axl = (c.i > 0) ? ax[n - 1] : 0.0;
        const size_t nl = (c.i > 0) ? n - 1 : n, nr = (c.i + 2 < g.nx) ? n + 2 : n + 1;
        const size_t nym = (c.j > 0) ? n - g.nx : n, nyp = (c.j < g.ny - 1) ? n + g.nx : n;
        const double2 AYm = (c.j > 0) ? ld2(ay + nym) : make_double2(0.0, 0.0);
        const double Fl = F[nl], Kl = kappa[nl], Fr = F[nr], Kr = kappa[nr];
        const double2 Fym = ld2(F + nym), Kym = ld2(kappa + nym), Fyp = ld2(F + nyp),
                      Kyp = ld2(kappa + nyp);
        const double2 Fzm = ld2(F + c.nzm), Kzm = ld2(kappa + c.nzm), Fzp = ld2(F + c.nzp),
                      Kzp = ld2(kappa + c.nzp);
        double2 out;
        {   // left cell (i): x- neighbour nl, x+ neighbour the right cell
            const double t0 = ssf_term(axl, sigma, Kc.x, Kl, Fc.x, Fl);
            const double t1 = ssf_term(AX.x, sigma, Kc.x, Kc.y, Fc.x, Fc.y);
            const double t2 = ssf_term(AYm.x, sigma, Kc.x, Kym.x, Fc.x, Fym.x);
            const double t3 = ssf_term(AY.x, sigma, Kc.x, Kyp.x, Fc.x, Fyp.x);
            const double t4 = ssf_term(AZm.x, sigma, Kc.x, Kzm.x, Fc.x, Fzm.x);
            const double t5 = ssf_term(AZ.x, sigma, Kc.x, Kzp.x, Fc.x, Fzp.x);
            out.x = -(((((t0 + t1) + t2) + t3) + t4) + t5);
        }
        {   // right cell (i+1): x- neighbour the left cell, x+ neighbour nr (itself at the wall)
            const double t0 = ssf_term(AX.x, sigma, Kc.y, Kc.x, Fc.y, Fc.x);
            const double t1 = ssf_term(AX.y, sigma, Kc.y, Kr, Fc.y, Fr);
            const double t2 = ssf_term(AYm.y, sigma, Kc.y, Kym.y, Fc.y, Fym.y);
            const double t3 = ssf_term(AY.y, sigma, Kc.y, Kyp.y, Fc.y, Fyp.y);
            const double t4 = ssf_term(AZm.y, sigma, Kc.y, Kzm.y, Fc.y, Fzm.y);
            const double t5 = ssf_term(AZ.y, sigma, Kc.y, Kzp.y, Fc.y, Fzp.y);
            out.y = -(((((t0 + t1) + t2) + t3) + t4) + t5);
        }
        *reinterpret_cast<double2 *>(rhs + n) = out;
    }
}

}  // namespace ps
