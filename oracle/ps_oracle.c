/*
 * ps_oracle.c -- CPU oracle for the variable-coefficient pressure-Poisson red-black SOR path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path under paper_2104_01636_b200/csrc/.
 *
 * What it is: the method is an ITERATION, so the oracle is the algorithm written out step by
 * step in the order of SURVEY.md §8.c O1-O6, plain triple loops, fp64, no blocking, no fusion,
 * no reordering.  Build: gcc -O2 -ffp-contract=off (no FMA contraction, no fast-math), so every
 * expression below rounds exactly as written.
 *
 * Paper passages followed (citations are lines of /root/reference/PAPER.md):
 *   O1 density           rho = alpha*rho_l + (1-alpha)*rho_g        PAPER.md:66 eq (4), :92 step 4
 *   O2 face coefficient  linear averaging c->f of rho, then 1/rho_f PAPER.md:117; operator :111
 *      boundaries        no-penetration walls in x,y; periodic z
 *      grid              uniform Cartesian collocated
 *   O3/O4 red-black SOR  "red black SOR relaxation scheme"
 *   O5/O6 residual, L2 norms, stopping rule: the paper is silent; BASELINE.json north_star and
 *      DESIGN.md readings S1-S10 fix them.
 *
 * Pins (tests/test_oracle_pins.py, tests/golden/): closed-form eigenvalues of the constant-rho
 * operator (P1), dense LU on 4x4x8 (P2), symmetry (P3), flux telescoping / compatibility (P4),
 * 1-D periodic variable-coefficient closed form (P5), Gauss-Seidel zero residual on the updated
 * colour (P6), even z-shift bitwise invariance (P7), power-of-two scaling (P8), Young's SOR rate
 * (P9), energy monotonicity (P10).  Every function here is pinned by at least one of them.
 *
 * Layout: n = i + nx*(j + ny*k), x fastest, z slowest; all fields double.
 * Sign convention: (A p)_c = sum_f a_f (p_nb - p_c) = s - d*p_c; A p = rhs.
 */
#include <math.h>
#include <stddef.h>

#include "ps_oracle.h"

#define IDX(i, j, k) ((size_t)(i) + (size_t)nx * ((size_t)(j) + (size_t)ny * (size_t)(k)))

/* O1: eq (4).  F is the LIQUID volume fraction alpha. */
void ora_density(size_t n, const double *F, double rho_l, double rho_g, double *rho)
{
    for (size_t c = 0; c < n; ++c)
        rho[c] = (rho_l * F[c]) + (rho_g * (1.0 - F[c]));
}

/* O2: +x, +y, +z face coefficient of every cell, (1/h^2)/rho_f with rho_f the arithmetic mean of
 * the two cell densities ("linear averaging procedure to compute face value (eg.
 * rho_f ...)").  Wall faces are 0; z wraps ("periodic"). */
void ora_coefficients(int nx, int ny, int nz, double dx, double dy, double dz,
                      const double *rho, double *ax, double *ay, double *az)
{
    const double cx = 1.0 / (dx * dx), cy = 1.0 / (dy * dy), cz = 1.0 / (dz * dz);
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t n = IDX(i, j, k);
                ax[n] = (i < nx - 1) ? cx / (0.5 * (rho[n] + rho[IDX(i + 1, j, k)])) : 0.0;
                ay[n] = (j < ny - 1) ? cy / (0.5 * (rho[n] + rho[IDX(i, j + 1, k)])) : 0.0;
                az[n] = cz / (0.5 * (rho[n] + rho[IDX(i, j, (k + 1) % nz)]));
            }
}

/* The six face coefficients and neighbour values of cell (i,j,k), and the two sums of O3:
 *   s = sum_f a_f p_nb   (12 roundings, left to right)      d = sum_f a_f
 * A wall neighbour is read at the clamped index and multiplied by the 0.0 coefficient. */
static inline void stencil_sums(int nx, int ny, int nz, const double *ax, const double *ay,
                                const double *az, const double *p, int i, int j, int k,
                                double *s_out, double *d_out)
{
    const int km = (k - 1 + nz) % nz, kp = (k + 1) % nz;
    const double axm = (i > 0) ? ax[IDX(i - 1, j, k)] : 0.0;
    const double axp = ax[IDX(i, j, k)];
    const double aym = (j > 0) ? ay[IDX(i, j - 1, k)] : 0.0;
    const double ayp = ay[IDX(i, j, k)];
    const double azm = az[IDX(i, j, km)];
    const double azp = az[IDX(i, j, k)];
    const double pxm = p[IDX(i > 0 ? i - 1 : 0, j, k)];
    const double pxp = p[IDX(i < nx - 1 ? i + 1 : nx - 1, j, k)];
    const double pym = p[IDX(i, j > 0 ? j - 1 : 0, k)];
    const double pyp = p[IDX(i, j < ny - 1 ? j + 1 : ny - 1, k)];
    const double pzm = p[IDX(i, j, km)];
    const double pzp = p[IDX(i, j, kp)];
    *s_out = ((((axm * pxm + axp * pxp) + aym * pym) + ayp * pyp) + azm * pzm) + azp * pzp;
    *d_out = ((((axm + axp) + aym) + ayp) + azm) + azp;
}

/* O3: one half-sweep over the cells with ((i+j+k)&1) == colour ("red black SOR").
 * Cells of one colour never read each other, so the traversal order is free; OpenMP splits
 * the z planes and the result does not depend on the thread count. */
void ora_half_sweep(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                    const double *rhs, double *p, double omega, int colour)
{
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = (j + k + colour) & 1; i < nx; i += 2) {
                double s, d;
                stencil_sums(nx, ny, nz, ax, ay, az, p, i, j, k, &s, &d);
                const size_t n = IDX(i, j, k);
                const double g = (s - rhs[n]) / d;
                p[n] = p[n] + omega * (g - p[n]);
            }
}

/* O4: one sweep = red ((i+j+k) even) first, then black. */
void ora_sweep(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
               const double *rhs, double *p, double omega)
{
    ora_half_sweep(nx, ny, nz, ax, ay, az, rhs, p, omega, 0);
    ora_half_sweep(nx, ny, nz, ax, ay, az, rhs, p, omega, 1);
}

/* (A p)_c = s - d p_c: the discrete div(grad p / rho) of PAPER.md:111 (used by the pins). */
void ora_apply(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
               const double *p, double *Ap)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double s, d;
                stencil_sums(nx, ny, nz, ax, ay, az, p, i, j, k, &s, &d);
                const size_t n = IDX(i, j, k);
                Ap[n] = s - d * p[n];
            }
}

/* O5: r_c = rhs_c - (A p)_c; R2 = sum r^2, B2 = sum rhs^2, accumulated in long double in
 * linear-index order (serial on purpose). */
void ora_residual(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                  const double *rhs, const double *p, double *res_abs, double *res_rel,
                  double *rhs_norm)
{
    long double R2 = 0.0L, B2 = 0.0L;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double s, d;
                stencil_sums(nx, ny, nz, ax, ay, az, p, i, j, k, &s, &d);
                const size_t n = IDX(i, j, k);
                const double r = rhs[n] - (s - d * p[n]);
                R2 += (long double)r * (long double)r;
                B2 += (long double)rhs[n] * (long double)rhs[n];
            }
    const double ra = (double)sqrtl(R2), bn = (double)sqrtl(B2);
    *res_abs = ra;
    *rhs_norm = bn;
    *res_rel = (bn > 0.0) ? ra / bn : ra;
}

/* O6: sweeps s = 1..max_sweeps from the caller's p; if tol > 0 the residual is checked when
 * s % check_interval == 0 or s == max_sweeps and the loop stops at the first check with
 * ||r||/||rhs|| <= tol.  tol <= 0: exactly max_sweeps sweeps, norm computed once at the end. */
void ora_solve(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
               const double *rhs, double *p, double omega, int max_sweeps, double tol,
               int check_interval, ora_info *info)
{
    double ra = 0.0, rr = 0.0, bn = 0.0;
    int s = 0, converged = 0, checked = 0;
    for (s = 1; s <= max_sweeps; ++s) {
        ora_sweep(nx, ny, nz, ax, ay, az, rhs, p, omega);
        if (tol > 0.0 && (s % check_interval == 0 || s == max_sweeps)) {
            ora_residual(nx, ny, nz, ax, ay, az, rhs, p, &ra, &rr, &bn);
            checked = 1;
            if (rr <= tol) { converged = 1; break; }
        } else {
            checked = 0;
        }
    }
    if (s > max_sweeps) s = max_sweeps;
    if (!checked) ora_residual(nx, ny, nz, ax, ay, az, rhs, p, &ra, &rr, &bn);
    if (tol > 0.0 && rr <= tol) converged = 1;
    info->sweeps = s;
    info->converged = converged;
    info->res_abs = ra;
    info->res_rel = rr;
    info->rhs_norm = bn;
}

/* =====================================================================================
 * Multigrid acceleration of the red-black SOR ("multigrid accelerated red black SOR
 * relaxation scheme").  The paper gives no detail beyond those words, so
 * every choice below is a reading listed in DESIGN.md §12 (M1-M6): geometric cell-centred
 * coarsening by 2 in x, y and z, rediscretised coarse operator from averaged face coefficients,
 * 8-cell averaging restriction, piecewise-constant prolongation, red-black SOR as smoother and
 * as coarsest-level solver, V (gamma = 1) or W (gamma = 2) cycle.
 * Pins (tests/test_oracle_mg_pins.py): constant-rho coarse operator = the fine formula at 2h;
 * restriction/prolongation adjointness; coarse coefficients keep symmetry and zero row sums;
 * two-level cycle with an exact coarse solve reproduces the dense two-grid operator; the
 * converged result equals the dense LU solution; convergence factor of a constant-rho V-cycle.
 * ===================================================================================== */

/* M1: coarse face coefficient = 1/16 of the sum of the 4 fine face coefficients lying on the
 * coarse face (their arithmetic mean, times h^2/H^2 = 1/4).  Fine grid nx x ny x nz (all even),
 * coarse grid nx/2 x ny/2 x nz/2.  Wall faces stay 0 (the fine wall faces are 0), z wraps. */
void ora_mg_coarsen(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                    double *axc, double *ayc, double *azc)
{
    const int cx = nx / 2, cy = ny / 2, cz = nz / 2;
    for (int K = 0; K < cz; ++K)
        for (int J = 0; J < cy; ++J)
            for (int I = 0; I < cx; ++I) {
                const size_t c = (size_t)I + (size_t)cx * ((size_t)J + (size_t)cy * (size_t)K);
                const int i = 2 * I, j = 2 * J, k = 2 * K;
                axc[c] = 0.0625 * (((ax[IDX(i + 1, j, k)] + ax[IDX(i + 1, j + 1, k)])
                                    + ax[IDX(i + 1, j, k + 1)]) + ax[IDX(i + 1, j + 1, k + 1)]);
                ayc[c] = 0.0625 * (((ay[IDX(i, j + 1, k)] + ay[IDX(i + 1, j + 1, k)])
                                    + ay[IDX(i, j + 1, k + 1)]) + ay[IDX(i + 1, j + 1, k + 1)]);
                azc[c] = 0.0625 * (((az[IDX(i, j, k + 1)] + az[IDX(i + 1, j, k + 1)])
                                    + az[IDX(i, j + 1, k + 1)]) + az[IDX(i + 1, j + 1, k + 1)]);
            }
}

/* M2: residual field r = rhs - A p (the same expression as O5, stored). */
void ora_mg_residual_field(int nx, int ny, int nz, const double *ax, const double *ay,
                           const double *az, const double *rhs, const double *p, double *r)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double s, d;
                stencil_sums(nx, ny, nz, ax, ay, az, p, i, j, k, &s, &d);
                const size_t n = IDX(i, j, k);
                r[n] = rhs[n] - (s - d * p[n]);
            }
}

/* M3: restriction = mean of the 8 children, summed with x fastest, then y, then z. */
void ora_mg_restrict(int nx, int ny, int nz, const double *r, double *rc)
{
    const int cx = nx / 2, cy = ny / 2, cz = nz / 2;
    for (int K = 0; K < cz; ++K)
        for (int J = 0; J < cy; ++J)
            for (int I = 0; I < cx; ++I) {
                const int i = 2 * I, j = 2 * J, k = 2 * K;
                double t = r[IDX(i, j, k)] + r[IDX(i + 1, j, k)];
                t = t + r[IDX(i, j + 1, k)];
                t = t + r[IDX(i + 1, j + 1, k)];
                t = t + r[IDX(i, j, k + 1)];
                t = t + r[IDX(i + 1, j, k + 1)];
                t = t + r[IDX(i, j + 1, k + 1)];
                t = t + r[IDX(i + 1, j + 1, k + 1)];
                rc[(size_t)I + (size_t)cx * ((size_t)J + (size_t)cy * (size_t)K)] = 0.125 * t;
            }
}

/* M4: piecewise-constant prolongation, added to the fine iterate: p_c += e_parent(c). */
void ora_mg_prolong_add(int nx, int ny, int nz, const double *ec, double *p)
{
    const int cx = nx / 2, cy = ny / 2;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                p[IDX(i, j, k)] = p[IDX(i, j, k)]
                    + ec[(size_t)(i / 2) + (size_t)cx * ((size_t)(j / 2) + (size_t)cy * (size_t)(k / 2))];
}

/* M5: number of levels the grid allows: coarsen while nx, ny are even with nx/2, ny/2 >= 2 and
 * nz is a multiple of 4 (the coarse nz must stay even for the red-black colouring across the
 * periodic wrap). */
int ora_mg_max_levels(int nx, int ny, int nz)
{
    int L = 1;
    while (nx % 2 == 0 && ny % 2 == 0 && nz % 4 == 0 && nx / 2 >= 2 && ny / 2 >= 2) {
        nx /= 2; ny /= 2; nz /= 2; ++L;
    }
    return L;
}

typedef struct {
    int nx, ny, nz;
    double *ax, *ay, *az;   /* level 0: the caller's arrays */
    double *rhs, *p, *r;    /* level 0: rhs and p are the caller's */
} mg_level;

#include <stdlib.h>
#include <string.h>

/* M6: one cycle on level l.  Coarsest level: coarse_sweeps SOR sweeps.  Otherwise nu1 sweeps,
 * residual, restriction to the rhs of level l+1, zero initial guess there, gamma recursive
 * cycles (1 = V, 2 = W), prolongation added to p, nu2 sweeps.  On level l the smoothing counts are
 * min(nu * nu_growth^l, nu_max) (never below nu): coarse levels are cheap and the bubble modes
 * need them solved accurately (DESIGN.md §12 M6); from level 2 on the cap is
 * min(nu_max, nu_max_deep).  Every sweep of level 0 uses omega_s, every
 * sweep of a level l >= 1 (smoothing and the coarsest solve) omega_c. */
static int mg_nu(int nu, int l, const ora_mg_params *prm)
{
    /* the cap of level l: nu_max on level 1, min(nu_max, nu_max_deep) from level 2 on (the
     * bubble-offset modes are representable down to level 1 only: that is where
     * the sweeps pay; the levels below need fewer) */
    const int cap = (l >= 2 && prm->nu_max_deep < prm->nu_max) ? prm->nu_max_deep : prm->nu_max;
    long long v = nu;
    for (int q = 0; q < l && v < cap; ++q) v *= prm->nu_growth;
    return (int)(v < cap ? v : (nu < cap ? cap : nu));
}

static void mg_cycle(mg_level *lv, int l, int nlev, const ora_mg_params *prm)
{
    mg_level *f = &lv[l];
    const double omega = (l == 0) ? prm->omega_s : prm->omega_c;
    if (l == nlev - 1) {
        for (int s = 0; s < prm->coarse_sweeps; ++s)
            ora_sweep(f->nx, f->ny, f->nz, f->ax, f->ay, f->az, f->rhs, f->p, omega);
        return;
    }
    mg_level *c = &lv[l + 1];
    for (int s = 0, n1 = mg_nu(prm->nu1, l, prm); s < n1; ++s)
        ora_sweep(f->nx, f->ny, f->nz, f->ax, f->ay, f->az, f->rhs, f->p, omega);
    ora_mg_residual_field(f->nx, f->ny, f->nz, f->ax, f->ay, f->az, f->rhs, f->p, f->r);
    ora_mg_restrict(f->nx, f->ny, f->nz, f->r, c->rhs);
    memset(c->p, 0, sizeof(double) * (size_t)c->nx * c->ny * c->nz);
    for (int g = 0; g < prm->gamma; ++g) mg_cycle(lv, l + 1, nlev, prm);
    ora_mg_prolong_add(f->nx, f->ny, f->nz, c->p, f->p);
    for (int s = 0, n2 = mg_nu(prm->nu2, l, prm); s < n2; ++s)
        ora_sweep(f->nx, f->ny, f->nz, f->ax, f->ay, f->az, f->rhs, f->p, omega);
}

/* Multigrid solve: cycles c = 1..max_cycles from the caller's p, the O5 norm after every cycle,
 * stop at the first cycle with ||r||/||rhs|| <= tol (tol <= 0: exactly max_cycles cycles).
 * prm->levels is clipped to [1, ora_mg_max_levels].  info->sweeps returns the cycles done.
 * Returns 0, or -1 if memory ran out. */
int ora_mg_solve(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                 const double *rhs, double *p, const ora_mg_params *prm, int max_cycles,
                 double tol, ora_info *info)
{
    int nlev = prm->levels, maxl = ora_mg_max_levels(nx, ny, nz);
    if (nlev > maxl) nlev = maxl;
    if (nlev < 1) nlev = 1;
    mg_level lv[32];
    memset(lv, 0, sizeof lv);
    lv[0].nx = nx; lv[0].ny = ny; lv[0].nz = nz;
    lv[0].ax = (double *)ax; lv[0].ay = (double *)ay; lv[0].az = (double *)az;
    lv[0].rhs = (double *)rhs; lv[0].p = p;
    int ok = 1;
    for (int l = 0; l < nlev && ok; ++l) {
        const size_t n = (size_t)lv[l].nx * lv[l].ny * lv[l].nz;
        lv[l].r = (double *)malloc(n * sizeof(double));
        ok = ok && lv[l].r;
        if (l > 0) {
            lv[l].ax = (double *)malloc(n * sizeof(double));
            lv[l].ay = (double *)malloc(n * sizeof(double));
            lv[l].az = (double *)malloc(n * sizeof(double));
            lv[l].rhs = (double *)malloc(n * sizeof(double));
            lv[l].p = (double *)malloc(n * sizeof(double));
            ok = ok && lv[l].ax && lv[l].ay && lv[l].az && lv[l].rhs && lv[l].p;
            if (ok)
                ora_mg_coarsen(lv[l - 1].nx, lv[l - 1].ny, lv[l - 1].nz, lv[l - 1].ax, lv[l - 1].ay,
                               lv[l - 1].az, lv[l].ax, lv[l].ay, lv[l].az);
        }
        if (l + 1 < nlev) {
            lv[l + 1].nx = lv[l].nx / 2; lv[l + 1].ny = lv[l].ny / 2; lv[l + 1].nz = lv[l].nz / 2;
        }
    }
    double ra = 0.0, rr = 0.0, bn = 0.0;
    int c = 0, converged = 0;
    if (ok) {
        /* M7: the cycle is a fixed linear iteration; with omega_c close to 2 it can diverge on
         * operators it was not tuned on (strongly anisotropic spacing).  The only remedy taken is
         * the one stated in ora_mg_params: a lower omega_c for the cycles that follow. */
        ora_mg_params q = *prm;
        double best = 0.0;
        int have_best = 0, stall = 0;
        for (c = 1; c <= max_cycles; ++c) {
            mg_cycle(lv, 0, nlev, &q);
            ora_residual(nx, ny, nz, ax, ay, az, rhs, p, &ra, &rr, &bn);
            if (tol > 0.0 && rr <= tol) { converged = 1; break; }
            if (q.stall_cycles > 0) {
                if (!have_best || rr < best) {
                    best = rr; have_best = 1; stall = 0;
                } else if (++stall >= q.stall_cycles) {
                    q.omega_c = q.omega_c - q.omega_c_step;
                    if (q.omega_c < 1.0) q.omega_c = 1.0;
                    best = rr; stall = 0;
                }
            }
        }
        if (c > max_cycles) c = max_cycles;
        if (max_cycles == 0) ora_residual(nx, ny, nz, ax, ay, az, rhs, p, &ra, &rr, &bn);
    }
    for (int l = 0; l < nlev; ++l) {
        free(lv[l].r);
        if (l > 0) { free(lv[l].ax); free(lv[l].ay); free(lv[l].az); free(lv[l].rhs); free(lv[l].p); }
    }
    if (!ok) return -1;
    info->sweeps = c;
    info->converged = converged;
    info->res_abs = ra;
    info->res_rel = rr;
    info->rhs_norm = bn;
    return 0;
}

/* =====================================================================================
 * The steps either side of the solve: steps 10-12 of the paper's time
 * step.  Cell-centred intermediate velocity u^ = (ux, uy, uz); "c->f" is the
 * linear averaging of PAPER.md:117; walls in x, y carry no normal velocity (no-penetration,
 * PAPER.md:195), z is periodic.  Readings P1-P3 in DESIGN.md §13.
 * ===================================================================================== */

/* Face-normal velocities of cell (i,j,k): u^_f = u^_{c->f} (step 10), 0 on walls. */
static inline void face_velocities(int nx, int ny, int nz, const double *ux, const double *uy,
                                   const double *uz, int i, int j, int k, double f[6])
{
    const int km = (k - 1 + nz) % nz, kp = (k + 1) % nz;
    const size_t n = IDX(i, j, k);
    f[0] = (i > 0) ? 0.5 * (ux[IDX(i - 1, j, k)] + ux[n]) : 0.0;          /* x- */
    f[1] = (i < nx - 1) ? 0.5 * (ux[n] + ux[IDX(i + 1, j, k)]) : 0.0;     /* x+ */
    f[2] = (j > 0) ? 0.5 * (uy[IDX(i, j - 1, k)] + uy[n]) : 0.0;
    f[3] = (j < ny - 1) ? 0.5 * (uy[n] + uy[IDX(i, j + 1, k)]) : 0.0;
    f[4] = 0.5 * (uz[IDX(i, j, km)] + uz[n]);
    f[5] = 0.5 * (uz[n] + uz[IDX(i, j, kp)]);
}

/* Face values of (grad p / rho) . n of cell (i,j,k): a_f h (p_nb - p_c) with a_f = (1/h^2)/rho_f
 * the stored coefficient (0 on walls, where p is read at the clamped index). */
static inline void face_gradients(int nx, int ny, int nz, double dx, double dy, double dz,
                                  const double *ax, const double *ay, const double *az,
                                  const double *p, int i, int j, int k, double g[6])
{
    const int km = (k - 1 + nz) % nz, kp = (k + 1) % nz;
    const size_t n = IDX(i, j, k);
    const double pc = p[n];
    const double axm = (i > 0) ? ax[IDX(i - 1, j, k)] : 0.0;
    const double aym = (j > 0) ? ay[IDX(i, j - 1, k)] : 0.0;
    g[0] = (axm * dx) * (pc - p[IDX(i > 0 ? i - 1 : 0, j, k)]);
    g[1] = (ax[n] * dx) * (p[IDX(i < nx - 1 ? i + 1 : nx - 1, j, k)] - pc);
    g[2] = (aym * dy) * (pc - p[IDX(i, j > 0 ? j - 1 : 0, k)]);
    g[3] = (ay[n] * dy) * (p[IDX(i, j < ny - 1 ? j + 1 : ny - 1, k)] - pc);
    g[4] = (az[IDX(i, j, km)] * dz) * (pc - p[IDX(i, j, km)]);
    g[5] = (az[n] * dz) * (p[IDX(i, j, kp)] - pc);
}

/* P1 (step 11, right-hand side): rhs = div(u^_f) / dt. */
void ora_rhs_from_velocity(int nx, int ny, int nz, double dx, double dy, double dz,
                           const double *ux, const double *uy, const double *uz, double dt,
                           double *rhs)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double f[6];
                face_velocities(nx, ny, nz, ux, uy, uz, i, j, k, f);
                const double div = (((f[1] - f[0]) / dx) + ((f[3] - f[2]) / dy))
                                   + ((f[5] - f[4]) / dz);
                rhs[IDX(i, j, k)] = div / dt;
            }
}

/* P2 (step 12): u_c <- u^_c - dt (grad p / rho)_{f->c}, f->c the mean of the
 * two faces of the cell in each direction. */
void ora_correct_velocity(int nx, int ny, int nz, double dx, double dy, double dz,
                          const double *ax, const double *ay, const double *az, const double *p,
                          double dt, double *ux, double *uy, double *uz)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double g[6];
                face_gradients(nx, ny, nz, dx, dy, dz, ax, ay, az, p, i, j, k, g);
                const size_t n = IDX(i, j, k);
                ux[n] = ux[n] - dt * (0.5 * (g[0] + g[1]));
                uy[n] = uy[n] - dt * (0.5 * (g[2] + g[3]));
                uz[n] = uz[n] - dt * (0.5 * (g[4] + g[5]));
            }
}

/* P3: divergence of the corrected FACE velocity u_f = u^_f - dt (grad p / rho)_f, the quantity
 * the projection drives to zero: equals dt (rhs - A p) up to rounding. */
void ora_face_divergence(int nx, int ny, int nz, double dx, double dy, double dz, const double *ax,
                         const double *ay, const double *az, const double *ux, const double *uy,
                         const double *uz, const double *p, double dt, double *div)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double f[6], g[6], u[6];
                face_velocities(nx, ny, nz, ux, uy, uz, i, j, k, f);
                face_gradients(nx, ny, nz, dx, dy, dz, ax, ay, az, p, i, j, k, g);
                for (int q = 0; q < 6; ++q) u[q] = f[q] - dt * g[q];
                div[IDX(i, j, k)] = (((u[1] - u[0]) / dx) + ((u[3] - u[2]) / dy))
                                    + ((u[5] - u[4]) / dz);
            }
}

/* =====================================================================================
 * Second right-hand side through the same solver: the sharp-surface-force
 * pressure p~ of PAPER.md:70-78, eqs (6)-(7): sigma kappa n delta = -grad p~ enters
 * div(grad p~ / rho) = 0 "as a source term".  Reading (T1): n delta = grad alpha
 * (alpha = liquid fraction F), face curvature kappa_f by the linear c->f average,
 * so on every face (grad p~ / rho)_f = -sigma kappa_f (grad F / rho)_f and
 *     sum_f a_f (p~_nb - p~_c) = - sum_f a_f (sigma kappa_f) (F_nb - F_c)  =: rhs_c.
 * With an exact constant curvature the solution is p~ = sigma kappa (1 - F) + const: the jump
 * sigma kappa across the interface, and a face force balance that vanishes identically
 * ("spurious velocities ... reduce to machine zero").
 * ===================================================================================== */
void ora_ssf_rhs(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                 const double *F, const double *kappa, double sigma, double *rhs)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const int km = (k - 1 + nz) % nz, kp = (k + 1) % nz;
                const size_t n = IDX(i, j, k);
                const size_t nb[6] = {IDX(i > 0 ? i - 1 : 0, j, k), IDX(i < nx - 1 ? i + 1 : nx - 1, j, k),
                                      IDX(i, j > 0 ? j - 1 : 0, k), IDX(i, j < ny - 1 ? j + 1 : ny - 1, k),
                                      IDX(i, j, km), IDX(i, j, kp)};
                const double a[6] = {(i > 0) ? ax[nb[0]] : 0.0, ax[n], (j > 0) ? ay[nb[2]] : 0.0,
                                     ay[n], az[nb[4]], az[n]};
                double t[6];
                for (int q = 0; q < 6; ++q) {
                    const double kf = 0.5 * (kappa[n] + kappa[nb[q]]);
                    t[q] = (a[q] * (sigma * kf)) * (F[nb[q]] - F[n]);
                }
                rhs[n] = -(((((t[0] + t[1]) + t[2]) + t[3]) + t[4]) + t[5]);
            }
}
