/*
 * ps_poisson.h -- C ABI of libps_poisson.so: B200 (sm_100a) red-black SOR solver for the
 * variable-coefficient pressure Poisson equation of the projection step of Kumar & Vanka
 * (arXiv 2104.01636):
 *
 *        div( grad p / rho )^{n+1} = rhs                       PAPER.md:109-111 (§2.2 step 11)
 *        rho = alpha rho_l + (1 - alpha) rho_g                 PAPER.md:66 eq (4), :92 step 4
 *        face values by linear averaging c->f (rho_f)
 *        no-penetration walls in x and y, periodic z
 *        uniform Cartesian collocated grid
 *        "red black SOR relaxation scheme ... on a GPU"
 *
 * Everything the paper leaves open (omega, colour order, norm, stopping rule, wall treatment of
 * p) follows DESIGN.md "Readings" S1-S10.
 *
 * Conventions
 *   Grid nx x ny x nz, cell (i,j,k), linear index n = i + nx*(j + ny*k): x fastest, z slowest.
 *   All fields are fp64.  F is the LIQUID volume fraction (alpha of the paper).
 *   Discrete operator (A p)_c = sum_f a_f (p_nb - p_c), a_f = (1/h_f^2) / (0.5 (rho_c + rho_nb)),
 *   a_f = 0 on the x and y walls, z faces wrap.  One "sweep" = red half-sweep ((i+j+k) even)
 *   followed by black half-sweep = N cell updates:
 *        g = (sum_f a_f p_nb - rhs_c) / sum_f a_f ;   p_c <- p_c + omega (g - p_c).
 *
 * Pointers
 *   *_dev  : device memory owned by the caller (e.g. a torch tensor), contiguous natural layout,
 *            16-byte aligned, nx*ny*nz doubles.  Never freed or retained past the call.  A field
 *            pointer that is not 16-byte aligned is rejected with PS_EINVAL by every entry point
 *            (the kernels use 16-byte accesses and TMA; which kernel runs, and hence the
 *            summation tree of the norms, depends on the grid shape only, never on an address).
 *   *_host : host memory owned by the caller (pageable or pinned), same layout.
 *   Output scalars / ps_info are host pointers.
 *
 * Errors: every entry point returns 0 (PS_OK) or a negative code; nothing throws, aborts or
 * prints.  There is NO CPU fallback: without a CUDA device every compute call returns PS_ECUDA.
 * A ps_ctx is not thread-safe; distinct contexts are independent.
 */
#ifndef PS_POISSON_H
#define PS_POISSON_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

#define PS_OK       0
#define PS_EINVAL  (-1)   /* bad argument (see each call)                                  */
#define PS_ESTATE  (-2)   /* call order: solve/residual/sweeps before ps_set_fraction      */
#define PS_ECUDA   (-3)   /* a CUDA runtime call failed; ps_strerror gives the CUDA string */
#define PS_ENOMEM  (-4)   /* host or device allocation failed                              */
#define PS_ETOOBIG (-5)   /* ps_residual_noalloc: grid beyond PS_NOALLOC_MAX_CELLS           */

/* Sweep kernel variants (ps_set_kernel).  All give bitwise identical p. */
#define PS_KERNEL_AUTO     0   /* fastest variant the grid shape allows                     */
#define PS_KERNEL_TWOPASS  1   /* generic: one launch per colour, in place, any nx,ny>=1    */
#define PS_KERNEL_FUSED    2   /* red+black fused in one z-marching pass (both half-sweeps  */
                               /* temporally blocked in one launch), ping-pong p            */
#define PS_KERNEL_RESIDENT 3   /* L2-resident grids: n sweeps in ONE cooperative launch,    */
                               /* grid-wide barrier per half-sweep, in place, any nx,ny>=1  */
#define PS_KERNEL_FUSED_OTF 4  /* PS_KERNEL_FUSED with the face coefficients rebuilt in the  */
                               /* sweep from a stored rho field (O2 evaluated on the fly:   */
                               /* 32 instead of 48 B per cell-update, 8 more fp64 divisions */
                               /* per pair of updates).  Select it    */
                               /* BEFORE ps_set_fraction (which then also stores rho), else */
                               /* the sweeps return PS_ESTATE.                              */
#define PS_KERNEL_CLUSTER  5   /* grids that fit the shared memory of one thread-block      */
                               /* cluster (<= 16 CTAs x 227 KB: about 65 k cells): n sweeps */
                               /* in ONE launch, p and the coefficients on chip, z-slab     */
                               /* neighbours through distributed shared memory, one cluster */
                               /* barrier per half-sweep, in place, any nx,ny>=1            */

typedef struct ps_ctx ps_ctx;   /* opaque; one per grid */

typedef struct {
    int    sweeps;      /* sweeps performed by this call                                   */
    int    converged;   /* 1: tol > 0 and res_rel <= tol at the last check; else 0         */
    double res_abs;     /* || rhs - A p ||_2  (plain Euclidean, no 1/N)                    */
    double res_rel;     /* res_abs / ||rhs||_2   (res_abs itself if ||rhs||_2 == 0)        */
    double rhs_norm;    /* || rhs ||_2                                                     */
} ps_info;

/* Create a solver for the paper's problem statement: a uniform Cartesian collocated grid
 * (PAPER.md:45 §2, :199 §4) of nx x ny x nz cells with spacings dx,dy,dz, duct walls in x and y
 * and periodic z (§4), on the current CUDA device.
 * PS_EINVAL: out NULL; nx,ny < 1; nz < 2 or nz odd (the red-black colouring must stay
 * consistent across the periodic wrap); dx,dy,dz not finite or <= 0.
 * Allocates its own workspace (ps_workspace_bytes) with cudaMalloc unless ps_set_workspace
 * supplies one before the first ps_set_fraction. */
int ps_create(ps_ctx **out, int nx, int ny, int nz, double dx, double dy, double dz);

/* Free the context and any workspace the library allocated itself.  NULL is allowed. */
int ps_destroy(ps_ctx *c);

/* Bytes of device workspace the context needs: face coefficients ax, ay, az, the second p
 * buffer of the fused kernels, reduction partials and device scalars. */
size_t ps_workspace_bytes(const ps_ctx *c);

/* Hand the context a caller-owned device workspace (256-byte aligned, >= ps_workspace_bytes).
 * It is retained until ps_destroy or the next ps_set_workspace; coefficients built before the
 * switch are lost (ps_set_fraction must be called again).  PS_EINVAL if too small/misaligned. */
int ps_set_workspace(ps_ctx *c, void *ws_dev, size_t bytes);

/* CUDA stream (a cudaStream_t passed as void*) on which every later call enqueues its work.
 * Default: the legacy default stream (NULL). */
int ps_set_stream(ps_ctx *c, void *cuda_stream);

/* Residual check cadence K of ps_solve (default 50, K >= 1). */
int ps_set_check_interval(ps_ctx *c, int K);

/* Choose the sweep kernel (PS_KERNEL_*).  PS_EINVAL if the grid shape does not allow the
 * variant (the fused kernels need nx even). */
int ps_set_kernel(ps_ctx *c, int variant);
int ps_get_kernel(const ps_ctx *c);          /* the variant AUTO resolved to, or the one set */

/* Launch geometry of the fused kernel (tuning and tests; every setting gives bitwise identical p).
 * rows_per_thread: rows of the 64x16-cell box one thread updates per step; only 1 (16 row warps)
 * is built -- two rows per thread were measured slower on B200 throughout round 1 -- so 0 (keep)
 * and 1 are accepted.  z_chunks: 0 = the balanced split (the chunk count whose slowest CTA marches
 * the fewest planes; the items left over after the last full round of one item per SM are cut
 * again into equal z pieces, so that every CTA marches nearly the same number of planes);
 * n > 0 = every (x,y) tile cut into n z chunks, the tile x chunk items dealt round-robin to
 * the CTAs, no re-cut.
 * Synchronises the stream.  PS_EINVAL: fused kernel not available for this grid, values out of
 * range.  ps_get_tuning returns the setting, the number of tiles, of CTAs launched and of work
 * items (any output may be NULL). */
int ps_set_tuning(ps_ctx *c, int rows_per_thread, int z_chunks);
int ps_get_tuning(const ps_ctx *c, int *rows_per_thread, int *z_chunks, int *tiles, int *ctas,
                  int *items);

/* Two launch options of the fused kernel (every setting gives bitwise identical p; tests and A/B
 * measurements switch them):
 *   dependent_launch  1: every sweep after the first of a batch is launched with the
 *                     programmatic stream-serialisation attribute, so its CTAs set up and fetch
 *                     their first coefficient boxes while the previous sweep drains; 0: plain
 *                     stream order.
 *   pace_window       n > 0: no CTA issues a stage more than n stages ahead of the mean over all
 *                     CTAs of the launch, which keeps the halo rows and columns that neighbouring
 *                     tiles share inside L2 (one global counter, one atomic and one load per CTA
 *                     and four planes); 0: CTAs run free.
 * -1 (the default of both) leaves the choice to the library: dependent launches where a launch
 * is short (up to 96 z steps per CTA), pacing with a window of 2 where it is longer (it wins
 * cold bursts at full clocks, 5 % on the 34 M-cell and 24 % on the 151 M-cell duct, and is neutral
 * in sustained runs at the power cap).  ps_get_launch_options
 * returns the settings in effect.  PS_EINVAL: no fused kernel for this grid, values out of
 * range (pace_window > 64). */
int ps_set_launch_options(ps_ctx *c, int dependent_launch, int pace_window);
int ps_get_launch_options(const ps_ctx *c, int *dependent_launch, int *pace_window);

/* The work split of the fused kernel as a pure host computation (no device needed; host-logic
 * tests): tiles of an nx x ny x nz grid and the work items a launch on sm_count SMs would run,
 * z_chunks as in ps_set_tuning.  tiles_out: 4 ints per tile (xs, xe, ys, ye: owned cells
 * [xs,xe) x [ys,ye)), at most tile_cap tiles; items_out: 4 ints per item (cta, tile, ks, ke: CTA
 * `cta` marches tile `tile` over the planes [ks,ke)), in launch order, at most item_cap items;
 * either may be NULL.  The three counts are always returned.  PS_EINVAL: the fused kernel does
 * not take this grid (odd nx), bad arguments. */
int ps_fused_plan(int nx, int ny, int nz, int sm_count, int z_chunks, int *tiles_out, int tile_cap,
                  int *items_out, int item_cap, int *ntiles, int *nitems, int *nctas);

/* Step 4 of the paper's time step + face coefficients:
 * rho = rho_l F + rho_g (1-F); ax,ay,az = (1/h^2)/(0.5 (rho_c + rho_nb)) for the +x,+y,+z
 * face of every cell, 0 on the +x / +y wall faces, +z wraps.  One launch, asynchronous on
 * the stream.  F_dev is only read during the call.  PS_EINVAL: NULL, rho_l or rho_g <= 0 or
 * not finite.  Not checked on the device: F in [0,1], finite. */
int ps_set_fraction(ps_ctx *c, const double *F_dev, double rho_l, double rho_g);

/* Copy the face coefficients out in natural layout (device pointers, any may be NULL). */
int ps_export_coefficients(ps_ctx *c, double *ax_dev, double *ay_dev, double *az_dev);

/* Step 11 of the paper's time step, div(grad p / rho) = rhs (§2.2), by the
 * "red black SOR relaxation scheme" of PAPER.md:78 §2.1: red-black SOR on A p = rhs starting from
 * the caller's p (in/out).  omega, colour order, norm and stopping rule are readings S3-S5 of
 * DESIGN.md §2 (the paper gives none).
 *   for s = 1..max_sweeps { red; black; if (tol > 0 && (s % K == 0 || s == max_sweeps)) check }
 * stopping at the first check with ||r||_2/||rhs||_2 <= tol.  tol <= 0: exactly max_sweeps
 * sweeps, norm computed once at the end.  Synchronises the stream before returning; the only
 * device->host traffic are the 16-byte norm read-backs.  Hitting max_sweeps is not an error
 * (info->converged = 0).  info may be NULL.
 * PS_EINVAL: NULL rhs/p, omega not in (0,2), max_sweeps < 0.  PS_ESTATE: no coefficients. */
int ps_solve(ps_ctx *c, const double *rhs_dev, double *p_dev, double omega, int max_sweeps,
             double tol, ps_info *info);

/* Exactly n sweeps, enqueued asynchronously: no norm, no host synchronisation (the throughput
 * window of bench.py; time it with events on the stream). */
int ps_sweeps(ps_ctx *c, const double *rhs_dev, double *p_dev, double omega, int n);

/* One colour only (colour 0 = red = (i+j+k) even, 1 = black), in place, generic kernel;
 * asynchronous.  For parity tests of the half-sweep itself. */
int ps_half_sweep(ps_ctx *c, const double *rhs_dev, double *p_dev, double omega, int colour);

/* Residual of step 11's equation (the norm is reading S5 of DESIGN.md §2, the paper
 * states none): ||rhs - A p||_2 and its ratio to ||rhs||_2 by the deterministic two-pass reduction
 * (fixed partition, warp-shuffle tree, single-block fixed-order final pass; no atomics).
 * Synchronises the stream.  Outputs are host pointers; res_rel / rhs_norm may be NULL. */
int ps_residual(ps_ctx *c, const double *rhs_dev, const double *p_dev, double *res_abs,
                double *res_rel, double *rhs_norm);

/* ps_residual for callers that cannot allocate device memory.
 *
 * Who that is: this solver is meant to sit inside a flow solver's time step, and
 * the residual of step 11 is evaluated in every one of them.  Such a host program
 * usually hands the whole GPU to a memory pool of its own (a framework's caching allocator, an
 * arena sized at start-up to the 180 GB of the board).  Inside it a cudaMalloc may simply fail
 * because the pool already holds the memory, and cudaMalloc / cudaFree stall every stream of the
 * device while they run, which a time step that overlaps several streams cannot afford.  A plug-in
 * that is handed raw pointers and a stream, but no allocator, is in the same position.  Every other
 * entry point of this header needs a ps_ctx, and ps_create allocates (host memory, a pinned
 * read-back word, the fused kernel's plan); this one needs none.
 *
 * What it computes: out_dev[0] = ||rhs - A p||_2, out_dev[1] = that over ||rhs||_2 (the norm itself
 * if rhs == 0), out_dev[2] = ||rhs||_2, with A given by the caller's face coefficients (the
 * arrays ps_export_coefficients writes, or the caller's own in the same layout: +x, +y, +z face of
 * every cell, 0 on the +x / +y wall faces).  Same summation tree as ps_residual, so the three
 * numbers are bitwise the same.  All pointers are device pointers owned by the caller, the five
 * fields 16-byte aligned and nx*ny*nz doubles, out_dev 3 doubles, 8-byte aligned.  One memset node
 * and one kernel launch on cuda_stream (a cudaStream_t passed as void*, NULL = the legacy default
 * stream); the call does not synchronise, out_dev is valid once the stream has reached that point.
 *
 * Scratch: the per-chunk partial sums live in a fixed array inside the library image (1 MiB +
 * 256 B of device memory on every GPU that loads the library, held until the process exits), so
 * the call runs no cudaMalloc, cudaFree, cudaMallocHost or any other allocating routine.  The
 * price is a size limit: grids of more than PS_NOALLOC_MAX_CELLS cells (2^28: every BASELINE.json
 * config fits, the largest has 151 M) are refused with PS_ETOOBIG before anything is enqueued.
 * The first call on a device looks up the array's device address (that device must be current,
 * as for every later call on it); make that first call outside any stream capture.
 * All calls on one device share the array, which keeps what the last call left in it.  The one
 * word that must start at zero (the counter by which the last block to finish is found) is
 * cleared at the start of every call; the partial sums need no clearing, a call reads only the
 * slots it has just written.  Two calls that can overlap on the GPU (different streams without
 * an event between them, or two host threads on one device) race on the array and give garbage:
 * order them.
 * PS_EINVAL: NULL or misaligned pointer; nx, ny < 1; nz < 2 or odd.  PS_ETOOBIG: see above.
 * PS_ECUDA: a runtime call failed (no device, sticky error). */
#define PS_NOALLOC_MAX_CELLS 268435456LL
int ps_residual_noalloc(int nx, int ny, int nz, const double *ax_dev, const double *ay_dev,
                        const double *az_dev, const double *rhs_dev, const double *p_dev,
                        void *cuda_stream, double *out_dev);

/* The whole path on HOST buffers (the end-to-end leg of bench.py): H2D of F and rhs and p,
 * ps_set_fraction, ps_solve, D2H of p.  The three device staging fields come from the caller's
 * ps_set_host_staging block (256-byte aligned, >= ps_host_staging_bytes, retained until
 * ps_destroy or replaced) or, without one, from a cudaMalloc on first use.  Same errors as the
 * calls it wraps. */
size_t ps_host_staging_bytes(const ps_ctx *c);
int ps_set_host_staging(ps_ctx *c, void *st_dev, size_t bytes);
int ps_solve_host(ps_ctx *c, const double *F_host, double rho_l, double rho_g,
                  const double *rhs_host, double *p_host, double omega, int max_sweeps,
                  double tol, ps_info *info);

/* Device-side timing of the sweep kernels, for the roofline line of bench.py.  When enabled,
 * every batch of sweep launches issued by ps_solve / ps_sweeps / ps_solve_host is bracketed by a
 * pair of CUDA events on the context's stream.  ps_timing synchronises the stream, adds up the
 * elapsed times since the last ps_timing call and returns them with the number of sweep-kernel
 * launches and the number of sweeps they cover (the resident kernel runs many sweeps per launch,
 * the two-pass kernel half a sweep); any output may be NULL. */
int ps_enable_timing(ps_ctx *c, int on);
int ps_timing(ps_ctx *c, double *sweep_ms, long long *sweep_launches, long long *sweeps);

/* ------------------------------------------------------------------------------------------
 * Multigrid acceleration of the red-black SOR ("multigrid accelerated red black SOR
 * relaxation scheme implemented on a GPU").  The paper gives no further
 * detail; DESIGN.md §12 lists the readings M1-M6: geometric coarsening by 2 in x, y, z while nx,
 * ny stay even and >= 2 after halving and nz is a multiple of 4; coarse face coefficient =
 * 1/16 of the sum of the 4 fine face coefficients on the coarse face; restriction = mean of the
 * 8 children of r = rhs - A p; piecewise-constant prolongation added to p; red-black SOR
 * (omega_s on the finest level, omega_c on every coarser one) as smoother (nu1 before, nu2
 * after; on level l multiplied by nu_growth^l up to nu_max -- min(nu_max, nu_max_deep) from
 * level 2 on --, because coarse levels are cheap and the bubble modes need level 1 solved
 * accurately) and as coarsest-level solver (coarse_sweeps);
 * gamma = 1 (V cycle) or 2 (W cycle). */
typedef struct {
    int levels;          /* requested levels, clipped to [1, what the grid allows]            */
    int nu1, nu2;        /* pre-/post-smoothing sweeps on the finest level (>= 0)              */
    int nu_growth;       /* level l smooths min(nu * nu_growth^l, nu_max) times (>= 1)         */
    int nu_max;          /* cap of the per-level count (>= 1; never lowers nu itself)          */
    int coarse_sweeps;   /* sweeps on the coarsest level (>= 1)                                */
    int gamma;           /* 1 = V, 2 = W                                                       */
    double omega_s;      /* relaxation factor of every sweep on level 0, in (0,2)              */
    double omega_c;      /* relaxation factor of every sweep on the levels l >= 1 (smoother    */
                         /* and coarsest solver), in (0,2)                                     */
    int nu_max_deep;     /* cap of the per-level count on the levels l >= 2 (>= 1; level 1 is  */
                         /* capped by nu_max alone; values >= nu_max change nothing)           */
    int stall_cycles;    /* safeguard of ps_mg_solve (M7), >= 0.  The cycle is a  */
                         /* fixed linear iteration and an omega_c close to 2 can diverge on     */
                         /* operators it was not tuned on (strongly anisotropic spacing).  > 0: */
                         /* once this many cycles in a row have ended with a norm that is not   */
                         /* below the best norm of the call so far, omega_c is lowered by       */
                         /* omega_c_step (never below 1) for the cycles that follow, that norm  */
                         /* becomes the new best and the count restarts.  0: never.  A          */
                         /* converging solve never triggers it; each ps_mg_solve call starts    */
                         /* from the omega_c of ps_mg_setup again                               */
    double omega_c_step; /* >= 0, finite                                                       */
} ps_mg_params;

/* Device memory of the coarse levels (per level: coefficients, ping-pong buffer, reduction
 * partials, right-hand side, correction).  ps_mg_workspace_bytes: bytes a hierarchy of `levels`
 * levels (clipped like ps_mg_setup clips them) needs.  ps_mg_set_workspace hands the context a
 * caller-owned block (256-byte aligned; retained until ps_destroy or replaced; any existing
 * hierarchy is dropped).  Without one the library allocates the block itself with cudaMalloc at
 * the first ps_mg_setup and frees it in ps_destroy. */
size_t ps_mg_workspace_bytes(const ps_ctx *c, int levels);
int ps_mg_set_workspace(ps_ctx *c, void *ws_dev, size_t bytes);

/* Build the level hierarchy from the coefficients of the last ps_set_fraction (one coarsening
 * launch per level).  Must be called again after every ps_set_fraction; the level contexts and
 * their memory are reused as long as the depth does not change.  On any failure the hierarchy is
 * dropped (ps_mg_levels() == 0) and ps_mg_solve returns PS_ESTATE until a set-up succeeds.
 * PS_EINVAL: bad parameters; a caller-owned level block that is too small; the current CUDA
 * device is not the one the context was created on.  PS_ESTATE: no coefficients. */
int ps_mg_setup(ps_ctx *c, const ps_mg_params *prm);
int ps_mg_levels(const ps_ctx *c);           /* levels in use (0 before ps_mg_setup) */

/* Multigrid cycles c = 1..max_cycles from the caller's p (in/out); after every cycle the
 * deterministic norm of ps_residual; stops at the first cycle with ||r||_2/||rhs||_2 <= tol
 * (tol <= 0: exactly max_cycles cycles).  info->sweeps returns the number of cycles.  When the
 * finest level has no pre-smoothing (nu1 = 0) the norm of a cycle is taken inside the residual +
 * restriction pass that opens the next one (same cycles, same p; the norm agrees with ps_residual
 * to rounding).  A cycle whose norm is not finite (a diverging parameter set, e.g. V(0,2) with
 * omega_s >= 1.85) ends the loop with converged = 0.
 * Synchronises the stream once per cycle (the norm read-back).  PS_ESTATE without ps_mg_setup. */
int ps_mg_solve(ps_ctx *c, const double *rhs_dev, double *p_dev, int max_cycles, double tol,
                ps_info *info);

/* The transfer operators on their own (parity tests): coarse coefficients of level 1 copied
 * out (nx/2 * ny/2 * nz/2 doubles each, any may be NULL); rc = restriction of rhs - A p. */
int ps_mg_export_coarse(ps_ctx *c, int level, double *ax_dev, double *ay_dev, double *az_dev);
int ps_mg_residual_restrict(ps_ctx *c, const double *rhs_dev, const double *p_dev, double *rc_dev);
int ps_mg_prolong_add(ps_ctx *c, const double *ec_dev, double *p_dev);

/* ------------------------------------------------------------------------------------------
 * The steps either side of the solve (steps 10-12 of the time step; SURVEY.md
 * §8.f NEXT-2; readings P1-P3 of DESIGN.md §13).  ux, uy, uz: cell-centred intermediate velocity
 * u^, device arrays in natural layout.  "c->f" is the linear averaging of PAPER.md:117; wall
 * faces carry no normal velocity, z is periodic.  All three are one asynchronous
 * launch on the context's stream.  PS_EINVAL: NULL pointer, dt <= 0 or not finite.
 * PS_ESTATE (correct / face divergence): no coefficients. */

/* rhs = div(u^_f) / dt  (right-hand side of step 11).  Needs no coefficients. */
int ps_rhs_from_velocity(ps_ctx *c, const double *ux_dev, const double *uy_dev,
                         const double *uz_dev, double dt, double *rhs_dev);

/* u_c <- u^_c - dt (grad p / rho)_{f->c}  (step 12), in place on ux, uy, uz. */
int ps_correct_velocity(ps_ctx *c, const double *p_dev, double dt, double *ux_dev, double *uy_dev,
                        double *uz_dev);

/* div_dev = div(u^_f - dt (grad p / rho)_f): the divergence of the corrected face velocity,
 * = dt (rhs - A p); what the projection drives to zero. */
int ps_face_divergence(ps_ctx *c, const double *ux_dev, const double *uy_dev, const double *uz_dev,
                       const double *p_dev, double dt, double *div_dev);

/* Right-hand side of the sharp-surface-force pressure p~ (eqs (6)-(7); SURVEY.md
 * §8.f NEXT-3; reading T1 of DESIGN.md §14): rhs_c = - sum_f a_f (sigma kappa_f)(F_nb - F_c) with
 * kappa_f the linear c->f average of the cell curvatures kappa_dev and F_dev the liquid fraction
 * the coefficients were built from.  The p~ system is then solved with ps_solve / ps_mg_solve on
 * the same coefficients (a second right-hand side per coefficient set).  One asynchronous launch.
 * PS_EINVAL: NULL pointer, sigma not finite.  PS_ESTATE: no coefficients. */
int ps_ssf_rhs(ps_ctx *c, const double *F_dev, const double *kappa_dev, double sigma,
               double *rhs_dev);

/* Self-checking build (libps_poisson_checked.so, compiled with -DPS_CHECKED; compute-sanitizer is
 * not available on the B200 pool, profiles/r02_sanitizer.md): the fused sweep kernel checks its
 * shared-memory addressing, TMA destinations, global stores and its mbarrier ring protocol and
 * counts violations instead of faulting.  ps_checked_build: 1 in that build, 0 in the product
 * build.  ps_debug_read: out_host[0] = violations counted since ps_create over this context and
 * its multigrid levels, out_host[1..5] = the first one (code, three details, CTA << 32 | thread);
 * all zero in the product build.  Synchronises the stream.
 * ps_debug_sabotage(c, 1) makes the checked kernel skip the red-barrier wait of its row warps (a
 * deliberately broken protocol, harmless to memory: the negative control of the checks);
 * ps_debug_sabotage(c, 2) makes CTA 0 of a paced launch never claim its stages in the pacing
 * counter, as if it were not resident: the other CTAs must give up waiting (after ~1 ms each) and
 * the launch must end with the right result.  PS_EINVAL in the product build. */
int ps_checked_build(void);
int ps_debug_read(ps_ctx *c, unsigned long long *out_host);
int ps_debug_sabotage(ps_ctx *c, int mode);

/* Bandwidth probe for the roofline line of bench.py, no part of the solve path: out[i] = sum over
 * r < reads of in[r*n + i], i < n, in one launch of `blocks` blocks of 512 threads with 16-byte
 * streaming accesses.  reads = 5 is the fused sweep's mix (p, ax, ay, az, rhs in; p out), reads = 1
 * a plain copy.  in_dev: reads*n doubles, out_dev: n doubles, both 16-byte aligned device memory of
 * the caller; n even.  Asynchronous on cuda_stream (a cudaStream_t as void*); time it with events.
 * PS_EINVAL: NULL / misaligned pointer, n odd or < 2, reads not in {1, 3, 5}, blocks < 1. */
int ps_stream_probe(const double *in_dev, double *out_dev, size_t n, int reads, int blocks,
                    void *cuda_stream);

/* Kernels launched by this context since ps_create (bench.py's gpu_launches). */
long long ps_launch_count(const ps_ctx *c);

/* Text for a return code; for PS_ECUDA the last CUDA error string seen by this thread. */
const char *ps_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
