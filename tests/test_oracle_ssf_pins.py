"""Pins of the oracle's sharp-surface-force right-hand side (eqs (6)-(7); reading
T1 of DESIGN.md §14).  What the paper fixes: the pressure jump across the interface is sigma kappa
and, with the exact curvature, the surface force is balanced identically ("spurious velocities
... reduce to machine zero for a static bubble with exact analytical curvature").
"""
import numpy as np

from paper_2104_01636_b200 import workload as wl


def setup(ora, nx=24, ny=24, nz=32, count=1, D=8, seed=3):
    w = wl.make_custom(nx, ny, nz, count, D, seed)
    coef = ora.coefficients(w.F, w.rho_l, w.rho_g, w.dx, w.dy, w.dz)
    kappa = wl.curvature_field(nx, ny, nz, w.centres, D, w.dx)
    return w, coef, kappa


def test_rhs_lives_on_the_interface_and_is_compatible(ora):
    w, coef, kappa = setup(ora)
    rhs = ora.ssf_rhs(coef, w.F, kappa, wl.SIGMA)
    nb_same = np.ones_like(w.F, dtype=bool)
    for ax in range(3):
        for s in (1, -1):
            nb_same &= np.roll(w.F, s, axis=ax) == w.F
    assert np.all(rhs[nb_same] == 0.0)                 # no jump in F, no source
    assert np.count_nonzero(rhs) > 0
    assert abs(rhs.sum()) <= 1e-12 * np.abs(rhs).sum()     # face terms telescope


def test_constant_curvature_rhs_is_minus_sigma_kappa_A_F(ora):
    w, coef, _ = setup(ora, count=2)
    kap = 2.0 / (4 * w.dx)
    rhs = ora.ssf_rhs(coef, w.F, np.full_like(w.F, kap), wl.SIGMA)
    want = -wl.SIGMA * kap * ora.apply(coef, w.F)
    assert np.max(np.abs(rhs - want)) <= 1e-12 * np.max(np.abs(want))


def test_static_bubble_pressure_jump_and_force_balance(ora):
    """Solve the p~ system: p~ = sigma kappa (1 - F) + const (Laplace jump sigma kappa = 2 sigma/R
    between gas and liquid), and the face force balance (grad p~ + sigma kappa grad F)/rho is zero
    on every face to solver tolerance -- the paper's "machine zero" spurious velocity."""
    w, coef, kappa = setup(ora)
    R = 4 * w.dx
    rhs = ora.ssf_rhs(coef, w.F, kappa, wl.SIGMA)
    p = np.zeros_like(rhs)
    info = ora.mg_solve(coef, rhs, p, 300, 1e-12, levels=3, nu1=2, nu2=2, coarse_sweeps=100,
                        omega_s=1.5, nu_growth=4, nu_max=16)
    assert info.converged
    want = wl.SIGMA * (2.0 / R) * (1.0 - w.F)
    d = (p - p.mean()) - (want - want.mean())
    assert np.max(np.abs(d)) <= 1e-8 * wl.SIGMA * 2.0 / R
    jump = p[w.F == 0.0].mean() - p[w.F == 1.0].mean()
    assert abs(jump - 2.0 * wl.SIGMA / R) <= 1e-8 * 2.0 * wl.SIGMA / R
    # face accelerations: z faces as a sample of the balance
    az = coef[2]
    acc = az * w.dz * ((np.roll(p, -1, axis=0) - p)
                       + wl.SIGMA * 0.5 * (kappa + np.roll(kappa, -1, axis=0))
                       * (np.roll(w.F, -1, axis=0) - w.F))
    assert np.max(np.abs(acc)) <= 1e-7 * np.max(np.abs(az * w.dz)) * wl.SIGMA * 2.0 / R


def test_curvature_generator(ora):
    w, _, kappa = setup(ora, count=3, D=8, nx=32, ny=32, nz=48)
    vals = np.unique(kappa)
    assert set(vals) == {0.0, 2.0 / (4 * w.dx)}
    assert np.all(kappa[w.F < 1.0] > 0.0)               # every interface/gas cell has its kappa
    nbr = np.zeros_like(w.F, dtype=bool)
    for ax in range(3):
        for s in (1, -1):
            nbr |= np.roll(w.F, s, axis=ax) < 1.0
    assert np.all(kappa[nbr] > 0.0)                     # and so has every face neighbour
