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

#ifdef __cplusplus
}
#endif
#endif
