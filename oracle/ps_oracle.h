/* ps_oracle.h -- declarations of the CPU oracle (TEST INFRASTRUCTURE; see ps_oracle.c).
 * Not shared with the CUDA path: include/ps_poisson.h is a separate, independent header. */
#ifndef PS_ORACLE_H
#define PS_ORACLE_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int sweeps;        /* sweeps performed */
    int converged;     /* 1 iff tol > 0 and ||r||/||rhs|| <= tol at the last check */
    double res_abs;    /* ||rhs - A p||_2 */
    double res_rel;    /* res_abs / ||rhs||_2 (res_abs if ||rhs||_2 == 0) */
    double rhs_norm;   /* ||rhs||_2 */
} ora_info;

void ora_density(size_t n, const double *F, double rho_l, double rho_g, double *rho);
void ora_coefficients(int nx, int ny, int nz, double dx, double dy, double dz,
                      const double *rho, double *ax, double *ay, double *az);
void ora_half_sweep(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                    const double *rhs, double *p, double omega, int colour);
void ora_sweep(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
               const double *rhs, double *p, double omega);
void ora_apply(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
               const double *p, double *Ap);
void ora_residual(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                  const double *rhs, const double *p, double *res_abs, double *res_rel,
                  double *rhs_norm);
void ora_solve(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
               const double *rhs, double *p, double omega, int max_sweeps, double tol,
               int check_interval, ora_info *info);

/* Multigrid acceleration (readings M1-M6 of DESIGN.md §12). */
typedef struct {
    int levels;          /* requested number of levels (clipped to what the grid allows) */
    int nu1, nu2;        /* pre- and post-smoothing sweeps on level 0 */
    int nu_growth;       /* level l smooths min(nu * nu_growth^l, nu_max) times (1 = same everywhere) */
    int nu_max;          /* cap of the per-level smoothing count */
    int coarse_sweeps;   /* SOR sweeps on the coarsest level */
    int gamma;           /* recursive cycles per level: 1 = V, 2 = W */
    double omega_s;      /* relaxation factor of the smoother on level 0 (and of the only level when
                          * levels = 1) */
    double omega_c;      /* relaxation factor on the coarse levels l >= 1: smoother and coarsest
                          * solver (DESIGN.md §12 M6) */
    int nu_max_deep;     /* cap of the per-level smoothing count on the levels l >= 2 (level 1 is
                          * capped by nu_max alone); values >= nu_max change nothing */
    int stall_cycles;    /* DESIGN.md §12 M7 (safeguard of ora_mg_solve, not part of a cycle): > 0:
                          * once this many cycles in a row have ended with a norm that is not below
                          * the best norm so far, omega_c is lowered by omega_c_step (never below
                          * 1) for the cycles that follow, that norm becomes the new best and the
                          * count restarts; 0: omega_c stays as given */
    double omega_c_step; /* >= 0 */
} ora_mg_params;

void ora_mg_coarsen(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                    double *axc, double *ayc, double *azc);
void ora_mg_residual_field(int nx, int ny, int nz, const double *ax, const double *ay,
                           const double *az, const double *rhs, const double *p, double *r);
void ora_mg_restrict(int nx, int ny, int nz, const double *r, double *rc);
void ora_mg_prolong_add(int nx, int ny, int nz, const double *ec, double *p);
int ora_mg_max_levels(int nx, int ny, int nz);
int ora_mg_solve(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                 const double *rhs, double *p, const ora_mg_params *prm, int max_cycles,
                 double tol, ora_info *info);

/* Steps 10-12 of the paper's time step around the solve. */
void ora_rhs_from_velocity(int nx, int ny, int nz, double dx, double dy, double dz,
                           const double *ux, const double *uy, const double *uz, double dt,
                           double *rhs);
void ora_correct_velocity(int nx, int ny, int nz, double dx, double dy, double dz,
                          const double *ax, const double *ay, const double *az, const double *p,
                          double dt, double *ux, double *uy, double *uz);
void ora_face_divergence(int nx, int ny, int nz, double dx, double dy, double dz, const double *ax,
                         const double *ay, const double *az, const double *ux, const double *uy,
                         const double *uz, const double *p, double dt, double *div);

/* Sharp-surface-force right-hand side for p~ (eqs (6)-(7)). */
void ora_ssf_rhs(int nx, int ny, int nz, const double *ax, const double *ay, const double *az,
                 const double *F, const double *kappa, double sigma, double *rhs);

#ifdef __cplusplus
}
#endif
#endif
