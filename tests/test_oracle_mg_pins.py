"""Pins of the oracle's multigrid steps M1-M6 ("multigrid accelerated red black SOR";
readings in DESIGN.md §12).  The paper gives no multigrid detail, so the pins are what the
mathematics fixes: the coarse operator of a constant-density problem is the fine formula at 2h,
the Galerkin relation R A P = 2 A_c that ties coarsening, restriction and prolongation to the
(already pinned) fine operator, adjointness of R and P, symmetry and zero row sums of every
coarse operator, reduction to plain SOR with one level, convergence to the dense LU solution,
and textbook convergence behaviour of a constant-coefficient V-cycle.
"""
import numpy as np
import pytest

from paper_2104_01636_b200 import workload as wl


def rnd(shape, seed, stream=9):
    n = int(np.prod(shape))
    return (2.0 * wl.uniform01(seed, stream, np.arange(n, dtype=np.uint64)) - 1.0).reshape(shape)


def var_coef(ora, nx, ny, nz, seed, h=(0.1, 0.07, 0.13)):
    F = wl.random_fraction(nx, ny, nz, seed)
    return ora.coefficients(F, 1000.0, 1.2, *h)


# ------------------------------------------------------------------ M1
@pytest.mark.parametrize("Fval", [1.0, 0.25])
def test_coarse_operator_of_constant_density_is_the_2h_formula(ora, Fval):
    nx, ny, nz, dx, dy, dz = 8, 12, 16, 0.1, 0.07, 0.13
    fine = ora.coefficients(np.full((nz, ny, nx), Fval), 1000.0, 1.2, dx, dy, dz)
    want = ora.coefficients(np.full((nz // 2, ny // 2, nx // 2), Fval), 1000.0, 1.2,
                            2 * dx, 2 * dy, 2 * dz)
    got = ora.mg_coarsen(fine)
    for g, w in zip(got, want):
        assert np.max(np.abs(g - w)) <= 4e-16 * np.max(np.abs(w))
    assert np.all(got[0][:, :, -1] == 0.0) and np.all(got[1][:, -1, :] == 0.0)   # walls stay closed
    assert np.all(got[2] > 0.0)                                                   # z wraps


def test_galerkin_relation_ties_transfer_and_coarsening_to_the_fine_operator(ora):
    """For a coarse field E: restrict(A_f prolong(E)) = 2 A_c E  (fluxes through the 4 fine faces
    of every coarse face add up; R = 1/8 sum, a_F = 1/16 sum).  A wrong face index, weight or
    child order in M1, M3 or M4 breaks it."""
    nx, ny, nz = 8, 6, 12
    fine = var_coef(ora, nx, ny, nz, 3)
    coarse = ora.mg_coarsen(fine)
    E = rnd((nz // 2, ny // 2, nx // 2), 5)
    PE = np.zeros((nz, ny, nx))
    ora.mg_prolong_add(E, PE)
    lhs = ora.mg_restrict(ora.apply(fine, PE))
    rhs = 2.0 * ora.apply(coarse, E)
    assert np.max(np.abs(lhs - rhs)) <= 1e-13 * np.max(np.abs(rhs))


def test_coarse_operators_stay_symmetric_with_zero_row_sums(ora):
    coef = var_coef(ora, 16, 8, 16, 11)
    for _ in range(2):
        coef = ora.mg_coarsen(coef)
        shape = coef[0].shape
        x, y = rnd(shape, 1), rnd(shape, 2)
        a, b = float(np.sum(x * ora.apply(coef, y))), float(np.sum(y * ora.apply(coef, x)))
        assert abs(a - b) <= 1e-13 * max(abs(a), abs(b))
        ones = ora.apply(coef, np.ones(shape))
        assert np.max(np.abs(ones)) <= 1e-12 * np.max(coef[2])


# ------------------------------------------------------------------ M2
def test_residual_field_is_rhs_minus_apply_and_matches_the_norm(ora):
    nx, ny, nz = 10, 6, 8
    coef = var_coef(ora, nx, ny, nz, 4)
    rhs, p = rnd((nz, ny, nx), 6), rnd((nz, ny, nx), 7)
    r = ora.mg_residual_field(coef, rhs, p)
    assert np.max(np.abs(r - (rhs - ora.apply(coef, p)))) <= 1e-12 * np.max(np.abs(r))
    res_abs = ora.residual(coef, rhs, p)[0]
    assert abs(np.linalg.norm(r) - res_abs) <= 1e-13 * res_abs


# ------------------------------------------------------------------ M3, M4
def test_transfer_operators_constants_sums_and_adjointness(ora):
    nx, ny, nz = 6, 10, 8
    r = rnd((nz, ny, nx), 8)
    rc = ora.mg_restrict(r)
    assert rc.shape == (nz // 2, ny // 2, nx // 2)
    assert abs(8.0 * rc.sum() - r.sum()) <= 1e-13 * np.abs(r).sum()
    assert np.all(ora.mg_restrict(np.full((nz, ny, nx), 3.5)) == 3.5)
    p = np.full((nz, ny, nx), 1.0)
    ora.mg_prolong_add(np.full(rc.shape, 2.0), p)
    assert np.all(p == 3.0)
    e = rnd(rc.shape, 9)
    Pe = np.zeros((nz, ny, nx))
    ora.mg_prolong_add(e, Pe)
    assert abs(8.0 * np.sum(rc * e) - np.sum(r * Pe)) <= 1e-13 * np.sum(np.abs(r * Pe))
    # a single coarse value lands on exactly its 8 children
    e1 = np.zeros(rc.shape)
    e1[1, 2, 1] = 1.0
    P1 = np.zeros((nz, ny, nx))
    ora.mg_prolong_add(e1, P1)
    assert P1.sum() == 8.0 and np.all(P1[2:4, 4:6, 2:4] == 1.0)


# ------------------------------------------------------------------ M5
def test_level_count_rule(ora):
    assert ora.mg_max_levels(256, 256, 512) == 8       # 2x2x4 at the bottom
    assert ora.mg_max_levels(32, 32, 64) == 5
    assert ora.mg_max_levels(16, 12, 20) == 2          # nz = 20 -> 10 (even), then 10 % 4 != 0
    assert ora.mg_max_levels(5, 7, 6) == 1
    assert ora.mg_max_levels(4, 4, 6) == 1             # coarse nz would be odd


# ------------------------------------------------------------------ M6
def test_one_level_cycle_is_plain_sor(ora):
    nx, ny, nz = 8, 8, 8
    coef = var_coef(ora, nx, ny, nz, 12)
    rhs = wl.remove_mean(rnd((nz, ny, nx), 13))
    p1, p2 = np.zeros_like(rhs), np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, p1, 3, 0.0, levels=1, coarse_sweeps=7, omega_s=1.3)
    ora.sweep(coef, rhs, p2, 1.3, 21)
    assert np.array_equal(p1, p2)


@pytest.mark.parametrize("gamma", [1, 2])
def test_mg_converges_to_the_dense_lu_solution(ora, gamma):
    nx, ny, nz = 4, 4, 8
    N = nx * ny * nz
    coef = var_coef(ora, nx, ny, nz, 21, h=(0.25, 0.25, 0.125))
    rhs = wl.remove_mean(rnd((nz, ny, nx), 22))
    A = np.empty((N, N))
    for n in range(N):                                   # columns of A through the pinned operator
        e = np.zeros(N)
        e[n] = 1.0
        A[:, n] = ora.apply(coef, e.reshape(nz, ny, nx)).reshape(-1)
    x = np.linalg.solve(A - np.ones((N, N)) / N, rhs.reshape(-1))
    p = np.zeros_like(rhs)
    info = ora.mg_solve(coef, rhs, p, 200, 1e-13, levels=2, nu1=2, nu2=2, coarse_sweeps=60,
                        gamma=gamma, omega_s=1.2)
    assert info.converged and info.res_rel <= 1e-13
    q = p.reshape(-1) - p.mean()
    assert np.max(np.abs(q - (x - x.mean()))) <= 1e-10 * np.max(np.abs(x))


def test_constant_density_v_cycle_converges_at_a_grid_independent_rate(ora):
    """Textbook multigrid behaviour: with constant coefficients the residual reduction per V(2,2)
    cycle is bounded well below 1 and does not degrade when the grid is refined (plain SOR's
    rate tends to 1 like 1 - O(h^2))."""
    factors = []
    for nx, ny, nz in ((16, 16, 32), (32, 32, 64)):
        coef = ora.coefficients(np.ones((nz, ny, nx)), 1000.0, 1.2, 1 / nx, 1 / nx, 1 / nx)
        rhs = wl.remove_mean(rnd((nz, ny, nx), 31))
        p = np.zeros_like(rhs)
        res = [1.0]
        for _ in range(8):
            res.append(ora.mg_solve(coef, rhs, p, 1, 0.0, levels=99, nu1=2, nu2=2,
                                    coarse_sweeps=30, gamma=1, omega_s=1.0).res_rel)
        assert all(b < a for a, b in zip(res, res[1:]))
        factors.append((res[-1] / res[3]) ** (1.0 / 5))
    assert max(factors) < 0.5
    assert factors[1] < factors[0] * 1.25


def test_mg_needs_far_fewer_passes_than_sor_on_a_bubbly_duct(ora):
    w = wl.make_custom(32, 32, 64, 2, 8, 7)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p = np.zeros_like(w.rhs)
    info = ora.mg_solve(coef, w.rhs, p, 60, 1e-8, levels=3, nu1=2, nu2=2, coarse_sweeps=200,
                        gamma=1, omega_s=1.2)
    assert info.converged and info.sweeps <= 60       # plain SOR: thousands of sweeps (config 1)
    assert abs(ora.residual(coef, w.rhs, p)[1] - info.res_rel) <= 1e-12 * info.res_rel


def test_level_dependent_smoothing_counts(ora):
    """nu_growth = 1 is the plain cycle; with growth the coarse levels get min(nu g^l, nu_max)
    sweeps: two levels with nu_growth = 3 equal two levels whose coarsest solver runs the same
    number of sweeps -- checked through a case where level 1 IS the coarsest (growth must not
    touch coarse_sweeps) and through a 3-level case against hand-unrolled oracle steps."""
    nx, ny, nz = 8, 8, 16
    coef = var_coef(ora, nx, ny, nz, 41)
    rhs = wl.remove_mean(rnd((nz, ny, nx), 42))
    a, b = np.zeros_like(rhs), np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, a, 2, 0.0, levels=2, nu1=1, nu2=1, coarse_sweeps=9, omega_s=1.3,
                 nu_growth=3, nu_max=100)
    ora.mg_solve(coef, rhs, b, 2, 0.0, levels=2, nu1=1, nu2=1, coarse_sweeps=9, omega_s=1.3)
    assert np.array_equal(a, b)
    # 3 levels, nu = 1, growth 3, cap 2: level 0 smooths 1, level 1 smooths min(3, 2) = 2
    p = np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, p, 1, 0.0, levels=3, nu1=1, nu2=1, coarse_sweeps=5, omega_s=1.3,
                 nu_growth=3, nu_max=2)
    c1 = ora.mg_coarsen(coef)
    c2 = ora.mg_coarsen(c1)
    q = np.zeros_like(rhs)
    ora.sweep(coef, rhs, q, 1.3, 1)
    r1 = ora.mg_restrict(ora.mg_residual_field(coef, rhs, q))
    e1 = np.zeros_like(r1)
    ora.sweep(c1, r1, e1, 1.3, 2)
    r2 = ora.mg_restrict(ora.mg_residual_field(c1, r1, e1))
    e2 = np.zeros_like(r2)
    ora.sweep(c2, r2, e2, 1.3, 5)
    ora.mg_prolong_add(e2, e1)
    ora.sweep(c1, r1, e1, 1.3, 2)
    ora.mg_prolong_add(e1, q)
    ora.sweep(coef, rhs, q, 1.3, 1)
    assert np.array_equal(p, q)


def test_coarse_levels_relax_with_omega_c(ora):
    """M6: omega_s relaxes level 0 only, omega_c every level below it (smoothing and the coarsest
    solve) -- a 3-level V(1,2) cycle against hand-unrolled oracle steps with two different
    factors; omega_c = None is the one-factor cycle; one level never sees omega_c."""
    nx, ny, nz = 8, 8, 16
    coef = var_coef(ora, nx, ny, nz, 51)
    rhs = wl.remove_mean(rnd((nz, ny, nx), 52))
    w0, wc = 1.15, 1.85
    p = np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, p, 1, 0.0, levels=3, nu1=1, nu2=2, coarse_sweeps=5, omega_s=w0,
                 omega_c=wc, nu_growth=2, nu_max=100)
    c1 = ora.mg_coarsen(coef)
    c2 = ora.mg_coarsen(c1)
    q = np.zeros_like(rhs)
    ora.sweep(coef, rhs, q, w0, 1)
    r1 = ora.mg_restrict(ora.mg_residual_field(coef, rhs, q))
    e1 = np.zeros_like(r1)
    ora.sweep(c1, r1, e1, wc, 2)
    r2 = ora.mg_restrict(ora.mg_residual_field(c1, r1, e1))
    e2 = np.zeros_like(r2)
    ora.sweep(c2, r2, e2, wc, 5)
    ora.mg_prolong_add(e2, e1)
    ora.sweep(c1, r1, e1, wc, 4)
    ora.mg_prolong_add(e1, q)
    ora.sweep(coef, rhs, q, w0, 2)
    assert np.array_equal(p, q)
    # swapping the two factors is a different iteration (the pin would not see a cycle that
    # ignored omega_c or used it on level 0)
    s = np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, s, 1, 0.0, levels=3, nu1=1, nu2=2, coarse_sweeps=5, omega_s=wc,
                 omega_c=w0, nu_growth=2, nu_max=100)
    assert not np.array_equal(s, p)
    a, b = np.zeros_like(rhs), np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, a, 2, 0.0, levels=3, nu1=1, nu2=1, coarse_sweeps=5, omega_s=1.3)
    ora.mg_solve(coef, rhs, b, 2, 0.0, levels=3, nu1=1, nu2=1, coarse_sweeps=5, omega_s=1.3,
                 omega_c=1.3)
    assert np.array_equal(a, b)
    a, b = np.zeros_like(rhs), np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, a, 1, 0.0, levels=1, coarse_sweeps=7, omega_s=1.3, omega_c=0.7)
    ora.sweep(coef, rhs, b, 1.3, 7)
    assert np.array_equal(a, b)


def test_binding_defaults_converge_in_tens_of_cycles_in_the_oracle(ora):
    """The multigrid parameters the product uses by default (binding.MG_DEFAULTS: two relaxation
    factors, 48 sweeps per coarse level) run through the ORACLE's M1-M6 on config 1: the cycle
    converges to 1e-8 in about 16 cycles (SURVEY.md 8.f-1 "tens of cycles"; plain SOR needs 8,350
    sweeps), monotonically after the first cycles, and the solution satisfies the pinned operator."""
    from paper_2104_01636_b200 import binding          # constants only: no library is loaded
    w = wl.make_config(1)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    p = np.zeros_like(w.rhs)
    res = []
    for _ in range(40):
        info = ora.mg_solve(coef, w.rhs, p, 1, 0.0, **binding.MG_DEFAULTS)
        res.append(info.res_rel)
        if info.res_rel <= 1e-8:
            break
    assert res[-1] <= 1e-8 and 10 <= len(res) <= 24, (len(res), res[-1])
    assert all(b < a for a, b in zip(res[2:], res[3:]))
    r = w.rhs - ora.apply(coef, p)
    assert np.linalg.norm(r) <= 1.0001e-8 * np.linalg.norm(w.rhs)


def _cycle_by_hand(ora, coefs, l, rhs, p, post, coarse, w0, wc):
    """M6 spelled out from the oracle's step functions, V(0, post[l]) with an explicit list of
    post-smoothing counts per level (the schedule is what the test states, not a formula)."""
    w = w0 if l == 0 else wc
    if l == len(coefs) - 1:
        ora.sweep(coefs[l], rhs, p, w, coarse)
        return
    rc = ora.mg_restrict(ora.mg_residual_field(coefs[l], rhs, p))
    e = np.zeros_like(rc)
    _cycle_by_hand(ora, coefs, l + 1, rc, e, post, coarse, w0, wc)
    ora.mg_prolong_add(e, p)
    ora.sweep(coefs[l], rhs, p, w, post[l])


def test_deep_levels_have_their_own_cap(ora):
    """M6: the smoothing count of level l is min(nu g^l, nu_max) on level 1 and
    min(nu g^l, nu_max, nu_max_deep) from level 2 on.  Five levels on 32 x 32 x 64 with nu = 2,
    g = 3, nu_max = 7, nu_max_deep = 4: counts 2, 6, 4, 4 and 5 coarsest sweeps -- against the cycle
    assembled by hand from the oracle's steps with that list; nu_max_deep >= nu_max changes
    nothing; a cap that also bound level 1 (or none at all) gives another result."""
    nx, ny, nz = 32, 32, 64
    assert ora.mg_max_levels(nx, ny, nz) >= 5
    coef = var_coef(ora, nx, ny, nz, 61)
    rhs = wl.remove_mean(rnd((nz, ny, nx), 62))
    kw = dict(levels=5, nu1=0, nu2=2, coarse_sweeps=5, omega_s=1.3, omega_c=1.8, nu_growth=3, nu_max=7)
    coefs = [coef]
    for _ in range(4):
        coefs.append(ora.mg_coarsen(coefs[-1]))
    p = np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, p, 2, 0.0, nu_max_deep=4, **kw)
    q = np.zeros_like(rhs)
    for _ in range(2):
        _cycle_by_hand(ora, coefs, 0, rhs, q, [2, 6, 4, 4], 5, 1.3, 1.8)
    assert np.array_equal(p, q)
    a, b, c = np.zeros_like(rhs), np.zeros_like(rhs), np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, a, 2, 0.0, **kw)                          # no deep cap: 2, 6, 7, 7
    ora.mg_solve(coef, rhs, b, 2, 0.0, nu_max_deep=7, **kw)
    ora.mg_solve(coef, rhs, c, 2, 0.0, nu_max_deep=99, **kw)
    assert np.array_equal(a, b) and np.array_equal(a, c) and not np.array_equal(a, p)
    r = np.zeros_like(rhs)
    for _ in range(2):
        _cycle_by_hand(ora, coefs, 0, rhs, r, [2, 6, 7, 7], 5, 1.3, 1.8)
    assert np.array_equal(a, r)
    d = np.zeros_like(rhs)
    ora.mg_solve(coef, rhs, d, 2, 0.0, **dict(kw, nu_max=4))          # 2, 4, 4, 4: level 1 bound too
    assert not np.array_equal(d, p)


# ------------------------------------------------------------------ M7 (safeguard of the solve loop)
ANISO = dict(levels=6, nu1=0, nu2=2, coarse_sweeps=10, gamma=1, omega_s=1.4, omega_c=1.97,
             nu_growth=24, nu_max=48, nu_max_deep=48)


def _aniso_case(ora):
    w = wl.make_custom(16, 16, 32, 2, 8, 5, dx=4 / 16, dy=1 / 16, dz=1 / 16)   # spacing 4:1:1
    return w, ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)


def test_stall_safeguard_is_the_stated_bookkeeping_around_unchanged_cycles(ora):
    """M7 changes no cycle, only which omega_c the next one runs with.  One ora_mg_solve call with
    stall_cycles = 3, omega_c_step = 0.05 on a duct with 4:1:1 spacing (where omega_c = 1.97
    diverges) must equal, bitwise, single cycles (max_cycles = 1, safeguard off: the pinned
    cycle) strung together by hand with the rule as ora_mg_params states it: a norm below the best
    so far resets the count; the third norm in a row that is not lowers omega_c by the step, makes
    that norm the new best and restarts the count."""
    w, coef = _aniso_case(ora)
    ncyc = 30
    p = np.zeros_like(w.rhs)
    info = ora.mg_solve(coef, w.rhs, p, ncyc, 0.0, stall_cycles=3, omega_c_step=0.05, **ANISO)
    q = np.zeros_like(w.rhs)
    prm = dict(ANISO)
    best, stall, lowered, norms = None, 0, [], []
    for c in range(1, ncyc + 1):
        one = ora.mg_solve(coef, w.rhs, q, 1, 0.0, **prm)
        norms.append(one.res_rel)
        if best is None or one.res_rel < best:
            best, stall = one.res_rel, 0
        else:
            stall += 1
            if stall == 3:
                prm["omega_c"] = max(prm["omega_c"] - 0.05, 1.0)
                best, stall = one.res_rel, 0
                lowered.append(c)
    assert lowered, "the case must trigger the safeguard"
    assert lowered[0] >= 4                       # never before three non-improving norms
    assert np.array_equal(p, q)
    assert info.sweeps == ncyc and info.res_rel == norms[-1]
    # and it does what it is for: the plain cycle diverges here, the safeguarded one comes down
    r = np.zeros_like(w.rhs)
    plain = ora.mg_solve(coef, w.rhs, r, ncyc, 0.0, **ANISO)
    assert plain.res_rel > 1.0 > 0.05 > info.res_rel


def test_stall_safeguard_off_and_floor(ora):
    """stall_cycles = 0 is the cycle loop as it was (omega_c_step ignored); a converging run never
    triggers the safeguard (config-1-like duct, defaults: same p with and without); omega_c is
    never lowered below 1."""
    w, coef = _aniso_case(ora)
    a, b = np.zeros_like(w.rhs), np.zeros_like(w.rhs)
    ora.mg_solve(coef, w.rhs, a, 8, 0.0, **ANISO)
    ora.mg_solve(coef, w.rhs, b, 8, 0.0, stall_cycles=0, omega_c_step=0.5, **ANISO)
    assert np.array_equal(a, b)
    # floor: a step of 5 lands on omega_c = 1 after the first trigger, never below
    c, d = np.zeros_like(w.rhs), np.zeros_like(w.rhs)
    ora.mg_solve(coef, w.rhs, c, 12, 0.0, stall_cycles=1, omega_c_step=5.0, **ANISO)
    prm = dict(ANISO)
    best = None
    for _ in range(12):
        one = ora.mg_solve(coef, w.rhs, d, 1, 0.0, **prm)
        if best is None or one.res_rel < best:
            best = one.res_rel
        else:
            prm["omega_c"], best = 1.0, one.res_rel
    assert prm["omega_c"] == 1.0 and np.array_equal(c, d)
    # a healthy run: isotropic duct, nothing to safeguard
    v = wl.make_custom(16, 16, 32, 2, 8, 5)
    cv = ora.coefficients(v.F, v.rho_l, v.rho_g, v.dx, v.dy, v.dz)
    e, f = np.zeros_like(v.rhs), np.zeros_like(v.rhs)
    i1 = ora.mg_solve(cv, v.rhs, e, 40, 1e-8, **ANISO)
    i2 = ora.mg_solve(cv, v.rhs, f, 40, 1e-8, stall_cycles=3, omega_c_step=0.05, **ANISO)
    assert i1.converged and i2.converged and i1.sweeps == i2.sweeps and np.array_equal(e, f)
