"""ctypes wrapper around the CPU oracle (oracle/ps_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` legs may import this package.  Nothing under
paper_2104_01636_b200/ imports it, and it imports nothing from there.

`build()` compiles the C file with `gcc -O2 -ffp-contract=off -fopenmp` (no FMA contraction, no
fast-math).  Arrays are float64, C-contiguous, shape (nz, ny, nx).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ps_oracle.c")
_HDR = os.path.join(_HERE, "ps_oracle.h")
_LIB = os.path.join(_HERE, "libps_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/ps_oracle.c -> oracle/libps_oracle.so (no-op if up to date)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _LIB
    tmp = f"{_LIB}.{os.getpid()}.tmp"
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
           "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    os.replace(tmp, _LIB)
    return _LIB


class _Info(ctypes.Structure):
    _fields_ = [("sweeps", ctypes.c_int), ("converged", ctypes.c_int),
                ("res_abs", ctypes.c_double), ("res_rel", ctypes.c_double),
                ("rhs_norm", ctypes.c_double)]


@dataclass
class Info:
    sweeps: int
    converged: bool
    res_abs: float
    res_rel: float
    rhs_norm: float


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp, i, d, sz = ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        lib.ora_density.argtypes = [sz, dp, d, d, dp]
        lib.ora_coefficients.argtypes = [i, i, i, d, d, d, dp, dp, dp, dp]
        lib.ora_half_sweep.argtypes = [i, i, i, dp, dp, dp, dp, dp, d, i]
        lib.ora_sweep.argtypes = [i, i, i, dp, dp, dp, dp, dp, d]
        lib.ora_apply.argtypes = [i, i, i, dp, dp, dp, dp, dp]
        lib.ora_residual.argtypes = [i, i, i, dp, dp, dp, dp, dp, dp, dp, dp]
        lib.ora_solve.argtypes = [i, i, i, dp, dp, dp, dp, dp, d, i, d, i, ctypes.POINTER(_Info)]
        for f in ("ora_density", "ora_coefficients", "ora_half_sweep", "ora_sweep", "ora_apply",
                  "ora_residual", "ora_solve"):
            getattr(lib, f).restype = None
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"], "float64 C-contiguous expected"
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _shape(a: np.ndarray):
    nz, ny, nx = a.shape
    return nx, ny, nz


def density(F: np.ndarray, rho_l: float, rho_g: float) -> np.ndarray:
    F = np.ascontiguousarray(F, dtype=np.float64)
    rho = np.empty_like(F)
    _load().ora_density(F.size, _p(F), rho_l, rho_g, _p(rho))
    return rho


def coefficients(F: np.ndarray, rho_l: float, rho_g: float, dx: float, dy: float, dz: float):
    """O1 + O2: returns (ax, ay, az), each shaped like F."""
    rho = density(F, rho_l, rho_g)
    nx, ny, nz = _shape(rho)
    ax, ay, az = np.empty_like(rho), np.empty_like(rho), np.empty_like(rho)
    _load().ora_coefficients(nx, ny, nz, dx, dy, dz, _p(rho), _p(ax), _p(ay), _p(az))
    return ax, ay, az


def half_sweep(coef, rhs: np.ndarray, p: np.ndarray, omega: float, colour: int) -> None:
    ax, ay, az = coef
    nx, ny, nz = _shape(p)
    _load().ora_half_sweep(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(rhs), _p(p), omega, colour)


def sweep(coef, rhs: np.ndarray, p: np.ndarray, omega: float, count: int = 1) -> None:
    ax, ay, az = coef
    nx, ny, nz = _shape(p)
    lib = _load()
    for _ in range(count):
        lib.ora_sweep(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(rhs), _p(p), omega)


def apply(coef, p: np.ndarray) -> np.ndarray:
    ax, ay, az = coef
    nx, ny, nz = _shape(p)
    out = np.empty_like(p)
    _load().ora_apply(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(p), _p(out))
    return out


def residual(coef, rhs: np.ndarray, p: np.ndarray):
    """O5: returns (res_abs, res_rel, rhs_norm)."""
    ax, ay, az = coef
    nx, ny, nz = _shape(p)
    ra, rr, bn = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _load().ora_residual(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(rhs), _p(p),
                         ctypes.byref(ra), ctypes.byref(rr), ctypes.byref(bn))
    return ra.value, rr.value, bn.value


def solve(coef, rhs: np.ndarray, p: np.ndarray, omega: float, max_sweeps: int, tol: float,
          check_interval: int = 50) -> Info:
    """O6 in place on p."""
    ax, ay, az = coef
    nx, ny, nz = _shape(p)
    info = _Info()
    _load().ora_solve(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(rhs), _p(p), omega, max_sweeps,
                      tol, check_interval, ctypes.byref(info))
    return Info(info.sweeps, bool(info.converged), info.res_abs, info.res_rel, info.rhs_norm)


def threads() -> int:
    """OpenMP threads the half-sweeps use (OMP_NUM_THREADS or all cores)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env)
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


# ----------------------------------------------------------------------------- multigrid (M1-M6)
class _MgParams(ctypes.Structure):
    _fields_ = [("levels", ctypes.c_int), ("nu1", ctypes.c_int), ("nu2", ctypes.c_int),
                ("nu_growth", ctypes.c_int), ("nu_max", ctypes.c_int),
                ("coarse_sweeps", ctypes.c_int), ("gamma", ctypes.c_int),
                ("omega_s", ctypes.c_double), ("omega_c", ctypes.c_double),
                ("nu_max_deep", ctypes.c_int), ("stall_cycles", ctypes.c_int),
                ("omega_c_step", ctypes.c_double)]


def _mg_lib():
    lib = _load()
    if not getattr(lib, "_mg_ready", False):
        dp, i, d = ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double
        lib.ora_mg_coarsen.argtypes = [i, i, i, dp, dp, dp, dp, dp, dp]
        lib.ora_mg_residual_field.argtypes = [i, i, i, dp, dp, dp, dp, dp, dp]
        lib.ora_mg_restrict.argtypes = [i, i, i, dp, dp]
        lib.ora_mg_prolong_add.argtypes = [i, i, i, dp, dp]
        lib.ora_mg_max_levels.argtypes = [i, i, i]
        lib.ora_mg_max_levels.restype = i
        lib.ora_mg_solve.argtypes = [i, i, i, dp, dp, dp, dp, dp, ctypes.POINTER(_MgParams), i, d,
                                     ctypes.POINTER(_Info)]
        lib.ora_mg_solve.restype = i
        for f in ("ora_mg_coarsen", "ora_mg_residual_field", "ora_mg_restrict",
                  "ora_mg_prolong_add"):
            getattr(lib, f).restype = None
        lib._mg_ready = True
    return lib


def mg_coarsen(coef):
    """M1: coarse (ax, ay, az) on the nx/2 x ny/2 x nz/2 grid."""
    ax, ay, az = coef
    nx, ny, nz = _shape(ax)
    out = [np.empty((nz // 2, ny // 2, nx // 2)) for _ in range(3)]
    _mg_lib().ora_mg_coarsen(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(out[0]), _p(out[1]), _p(out[2]))
    return tuple(out)


def mg_residual_field(coef, rhs: np.ndarray, p: np.ndarray) -> np.ndarray:
    """M2: r = rhs - A p."""
    ax, ay, az = coef
    nx, ny, nz = _shape(p)
    r = np.empty_like(p)
    _mg_lib().ora_mg_residual_field(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(rhs), _p(p), _p(r))
    return r


def mg_restrict(r: np.ndarray) -> np.ndarray:
    """M3: mean of the 8 children."""
    nx, ny, nz = _shape(r)
    rc = np.empty((nz // 2, ny // 2, nx // 2))
    _mg_lib().ora_mg_restrict(nx, ny, nz, _p(r), _p(rc))
    return rc


def mg_prolong_add(ec: np.ndarray, p: np.ndarray) -> None:
    """M4: p += piecewise-constant interpolation of ec (in place)."""
    nx, ny, nz = _shape(p)
    _mg_lib().ora_mg_prolong_add(nx, ny, nz, _p(ec), _p(p))


def mg_max_levels(nx: int, ny: int, nz: int) -> int:
    return _mg_lib().ora_mg_max_levels(nx, ny, nz)


def mg_solve(coef, rhs: np.ndarray, p: np.ndarray, max_cycles: int, tol: float, levels: int = 99,
             nu1: int = 2, nu2: int = 2, coarse_sweeps: int = 50, gamma: int = 1,
             omega_s: float = 1.2, nu_growth: int = 1, nu_max: int = 1 << 20,
             omega_c: float | None = None, nu_max_deep: int | None = None,
             stall_cycles: int = 0, omega_c_step: float = 0.0) -> Info:
    """M5 + M6 in place on p; Info.sweeps holds the number of cycles.  omega_s relaxes level 0,
    omega_c the levels below it (None: the same factor everywhere); nu_max_deep caps the
    smoothing count from level 2 on (None: nu_max on every level); stall_cycles / omega_c_step:
    the safeguard M7 (0: off)."""
    ax, ay, az = coef
    nx, ny, nz = _shape(p)
    prm = _MgParams(levels, nu1, nu2, nu_growth, nu_max, coarse_sweeps, gamma, omega_s,
                    omega_s if omega_c is None else omega_c,
                    nu_max if nu_max_deep is None else nu_max_deep, stall_cycles, omega_c_step)
    info = _Info()
    rc = _mg_lib().ora_mg_solve(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(rhs), _p(p),
                                ctypes.byref(prm), max_cycles, tol, ctypes.byref(info))
    if rc != 0:
        raise MemoryError("ora_mg_solve")
    return Info(info.sweeps, bool(info.converged), info.res_abs, info.res_rel, info.rhs_norm)


# ----------------------------------------------------------------------------- steps 10-12 (P1-P3)
def _proj_lib():
    lib = _load()
    if not getattr(lib, "_proj_ready", False):
        dp, i, d = ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double
        lib.ora_rhs_from_velocity.argtypes = [i, i, i, d, d, d, dp, dp, dp, d, dp]
        lib.ora_correct_velocity.argtypes = [i, i, i, d, d, d, dp, dp, dp, dp, d, dp, dp, dp]
        lib.ora_face_divergence.argtypes = [i, i, i, d, d, d, dp, dp, dp, dp, dp, dp, dp, d, dp]
        for f in ("ora_rhs_from_velocity", "ora_correct_velocity", "ora_face_divergence"):
            getattr(lib, f).restype = None
        lib._proj_ready = True
    return lib


def rhs_from_velocity(u, h, dt: float) -> np.ndarray:
    """P1: rhs = div(u_f)/dt from the cell-centred (ux, uy, uz); h = (dx, dy, dz)."""
    ux, uy, uz = u
    nx, ny, nz = _shape(ux)
    rhs = np.empty_like(ux)
    _proj_lib().ora_rhs_from_velocity(nx, ny, nz, *h, _p(ux), _p(uy), _p(uz), dt, _p(rhs))
    return rhs


def correct_velocity(coef, p: np.ndarray, u, h, dt: float) -> None:
    """P2 in place on (ux, uy, uz)."""
    ax, ay, az = coef
    ux, uy, uz = u
    nx, ny, nz = _shape(p)
    _proj_lib().ora_correct_velocity(nx, ny, nz, *h, _p(ax), _p(ay), _p(az), _p(p), dt,
                                     _p(ux), _p(uy), _p(uz))


def face_divergence(coef, u, p: np.ndarray, h, dt: float) -> np.ndarray:
    """P3: divergence of the corrected face velocity."""
    ax, ay, az = coef
    ux, uy, uz = u
    nx, ny, nz = _shape(p)
    div = np.empty_like(p)
    _proj_lib().ora_face_divergence(nx, ny, nz, *h, _p(ax), _p(ay), _p(az), _p(ux), _p(uy), _p(uz),
                                    _p(p), dt, _p(div))
    return div


# ----------------------------------------------------------------------------- SSF rhs (T1)
def ssf_rhs(coef, F: np.ndarray, kappa: np.ndarray, sigma: float) -> np.ndarray:
    """rhs of the p~ system: -sum_f a_f (sigma kappa_f)(F_nb - F_c)."""
    ax, ay, az = coef
    nx, ny, nz = _shape(F)
    lib = _load()
    dp, i, d = ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double
    lib.ora_ssf_rhs.argtypes = [i, i, i, dp, dp, dp, dp, dp, d, dp]
    lib.ora_ssf_rhs.restype = None
    rhs = np.empty_like(F)
    lib.ora_ssf_rhs(nx, ny, nz, _p(ax), _p(ay), _p(az), _p(F), _p(kappa), sigma, _p(rhs))
    return rhs
