"""ctypes loader for the CPU fp64 ORACLE (oracle/mac_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares nothing with the CUDA path (paper_1910_12979_b200/).

All arithmetic is in mac_oracle.c; this file only marshals numpy arrays.  See mac_oracle.h for the
passages of PAPER.md each function follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libmac_oracle.so")
_SRC = os.path.join(_HERE, "mac_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "nodal_oracle.c")]          # one library: MAC projection + nodal projection
_HDRS = [os.path.join(_HERE, "mac_oracle.h"), os.path.join(_HERE, "nodal_oracle.h")]

PERIODIC, WALL, OUTFLOW = 0, 1, 2
PLANAR, SPHERICAL = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP on independent loops only)."""
    if (not force and os.path.exists(_LIB_PATH)
            and os.path.getmtime(_LIB_PATH) >= max(os.path.getmtime(p) for p in _SRCS + _HDRS)):
        return _LIB_PATH
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
           "-Wall", "-Wextra", "-o", _LIB_PATH, *_SRCS, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB_PATH


class Grid(C.Structure):
    _fields_ = [("n", C.c_int * 3), ("h", C.c_double * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3), ("rho_mean", C.c_int)]


class Base(C.Structure):
    _fields_ = [("geometry", C.c_int), ("nr", C.c_int), ("dr", C.c_double),
                ("center", C.c_double * 3)]


class MG(C.Structure):
    _fields_ = [("nu_pre", C.c_int), ("nu_post", C.c_int), ("max_cycles", C.c_int),
                ("rel_tol", C.c_double), ("coarsest_n", C.c_int), ("prolongation", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("cycles", C.c_int), ("singular", C.c_int), ("levels", C.c_int),
                ("converged", C.c_int), ("rhs_norm_inf", C.c_double),
                ("res_norm_inf", C.c_double), ("rhs_mean_removed", C.c_double),
                ("res_history", C.c_double * 128)]


_lib = None
_DP = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        # harness setting, not arithmetic: idle OpenMP threads sleep instead of spinning (the tiny
        # coarse-level loops otherwise stall for seconds when the host has fewer free cores than threads)
        os.environ.setdefault("OMP_WAIT_POLICY", "passive")
        L = C.CDLL(_LIB_PATH)
        GP, BP, MP = C.POINTER(Grid), C.POINTER(Base), C.POINTER(MG)
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_profile.restype = C.c_double
        L.orc_profile.argtypes = [_DP, C.c_int, C.c_double, C.c_double]
        L.orc_radius.restype = C.c_double
        L.orc_radius.argtypes = [BP, C.c_double, C.c_double, C.c_double]
        L.orc_face_coeff.argtypes = [GP, BP, _DP, _DP, _DP, _DP, _DP]
        L.orc_rho_from_profile.argtypes = [GP, BP, _DP, _DP]
        L.orc_make_beta0.argtypes = [C.c_int, _DP, _DP, _DP, _DP]
        L.orc_lateral_average.argtypes = [GP, BP, _DP, _DP, C.c_void_p]
        L.orc_dpdt_term.argtypes = [C.c_int, _DP, _DP, _DP, _DP]
        L.orc_effective_source.argtypes = [GP, BP, _DP, _DP, _DP]
        L.orc_rhs.argtypes = [GP, BP, _DP, _DP, _DP, _DP, _DP, _DP]
        L.orc_constraint.argtypes = [GP, BP, _DP, _DP, _DP, _DP, _DP, _DP]
        L.orc_norm_inf.restype = C.c_double
        L.orc_norm_inf.argtypes = [_DP, C.c_longlong]
        L.orc_mean.restype = C.c_double
        L.orc_mean.argtypes = [_DP, C.c_longlong]
        L.orc_shift.argtypes = [_DP, C.c_longlong, C.c_double]
        L.orc_is_singular.restype = C.c_int
        L.orc_is_singular.argtypes = [GP]
        L.orc_apply.argtypes = [GP, _DP, _DP, _DP, _DP, _DP]
        L.orc_diag.argtypes = [GP, _DP, _DP, _DP, _DP]
        L.orc_residual.argtypes = [GP, _DP, _DP, _DP, _DP, _DP, _DP]
        L.orc_rbgs_color.argtypes = [GP, _DP, _DP, _DP, _DP, _DP, C.c_int]
        L.orc_rbgs_sweep.argtypes = [GP, _DP, _DP, _DP, _DP, _DP]
        L.orc_can_coarsen.restype = C.c_int
        L.orc_can_coarsen.argtypes = [GP, C.c_int]
        L.orc_coarsen_grid.argtypes = [GP, GP]
        L.orc_coarsen_coeff.argtypes = [GP, _DP, _DP, _DP, _DP, _DP, _DP]
        L.orc_restrict.argtypes = [GP, _DP, _DP]
        L.orc_prolong_add.argtypes = [GP, _DP, _DP, C.c_int]
        L.orc_bottom_solve.restype = C.c_int
        L.orc_bottom_solve.argtypes = [GP, _DP, _DP, _DP, _DP, _DP]
        L.orc_vcycle.restype = C.c_int
        L.orc_vcycle.argtypes = [GP, _DP, _DP, _DP, _DP, _DP, MP]
        L.orc_correct.argtypes = [GP, _DP, _DP, _DP, _DP, _DP]
        L.orc_project.restype = C.c_int
        L.orc_project.argtypes = [GP, BP, MP, _DP, _DP, _DP, _DP, _DP, _DP, _DP, _DP,
                                  C.POINTER(Stats)]
        _lib = L
    return _lib


def _p(a):
    if a is None:
        return None
    assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(_DP)


def make_grid(n, h, bc_lo, bc_hi, rho_mean=0) -> Grid:
    g = Grid()
    g.rho_mean = int(rho_mean)
    for d in range(3):
        g.n[d], g.h[d], g.bc_lo[d], g.bc_hi[d] = int(n[d]), float(h[d]), int(bc_lo[d]), int(bc_hi[d])
    return g


def make_base(geometry, nr, dr, center=(0.0, 0.0, 0.0)) -> Base:
    b = Base()
    b.geometry, b.nr, b.dr = int(geometry), int(nr), float(dr)
    for d in range(3):
        b.center[d] = float(center[d])
    return b


def make_mg(nu_pre=2, nu_post=2, max_cycles=100, rel_tol=1e-10, coarsest_n=4, prolongation=0) -> MG:
    return MG(nu_pre, nu_post, max_cycles, rel_tol, coarsest_n, prolongation)


# Array shapes follow numpy C order with x fastest: cell arrays are [nz, ny, nx];
# u is [nz, ny, nx+1], v is [nz, ny+1, nx], w is [nz+1, ny, nx].

def cell_shape(g: Grid):
    return (g.n[2], g.n[1], g.n[0])


def face_shape(g: Grid, d: int):
    return (g.n[2] + (d == 2), g.n[1] + (d == 1), g.n[0] + (d == 0))


def coarsen_grid(g: Grid) -> Grid:
    c = Grid()
    lib().orc_coarsen_grid(C.byref(g), C.byref(c))
    return c


def profile(f, dr, r) -> float:
    return lib().orc_profile(_p(f), len(f), float(dr), float(r))


def face_coeff(g, b, beta0, rho):
    bx, by, bz = (np.empty(face_shape(g, d)) for d in range(3))
    lib().orc_face_coeff(C.byref(g), C.byref(b), _p(beta0), _p(rho), _p(bx), _p(by), _p(bz))
    return bx, by, bz


def rho_from_profile(g, b, rho0):
    rho = np.empty(cell_shape(g))
    lib().orc_rho_from_profile(C.byref(g), C.byref(b), _p(rho0), _p(rho))
    return rho


def lateral_average(g, b, rho):
    """O13.  Returns (rho0[nr], count[nr])."""
    rho0 = np.empty(b.nr)
    cnt = np.zeros(b.nr, dtype=np.int64)
    lib().orc_lateral_average(C.byref(g), C.byref(b), _p(rho), _p(rho0), cnt.ctypes.data_as(C.c_void_p))
    return rho0, cnt


def make_beta0(rho0, p0, gamma1bar):
    """O11 (Eq. 5)."""
    out = np.empty(len(rho0))
    lib().orc_make_beta0(len(rho0), _p(rho0), _p(p0), _p(gamma1bar), _p(out))
    return out


def dpdt_term(p0, gamma1bar, dp0dt):
    """O12: q = dp0dt / (Gamma1bar p0) on the samples (Eq. 6)."""
    out = np.empty(len(p0))
    lib().orc_dpdt_term(len(p0), _p(p0), _p(gamma1bar), _p(dp0dt), _p(out))
    return out


def effective_source(g, b, S, q):
    """O12: S - q(r_cell)."""
    out = np.empty(cell_shape(g))
    lib().orc_effective_source(C.byref(g), C.byref(b), _p(S), _p(q), _p(out))
    return out


def rhs(g, b, beta0, u, v, w, S=None):
    out = np.empty(cell_shape(g))
    lib().orc_rhs(C.byref(g), C.byref(b), _p(beta0), _p(u), _p(v), _p(w), _p(S), _p(out))
    return out


def constraint(g, b, beta0, u, v, w, S=None):
    out = np.empty(cell_shape(g))
    lib().orc_constraint(C.byref(g), C.byref(b), _p(beta0), _p(u), _p(v), _p(w), _p(S), _p(out))
    return out


def norm_inf(a) -> float:
    return lib().orc_norm_inf(_p(a), a.size)


def mean(a) -> float:
    return lib().orc_mean(_p(a), a.size)


def is_singular(g) -> bool:
    return bool(lib().orc_is_singular(C.byref(g)))


def apply(g, bx, by, bz, phi):
    out = np.empty(cell_shape(g))
    lib().orc_apply(C.byref(g), _p(bx), _p(by), _p(bz), _p(phi), _p(out))
    return out


def diag(g, bx, by, bz):
    out = np.empty(cell_shape(g))
    lib().orc_diag(C.byref(g), _p(bx), _p(by), _p(bz), _p(out))
    return out


def residual(g, bx, by, bz, phi, rhs_):
    out = np.empty(cell_shape(g))
    lib().orc_residual(C.byref(g), _p(bx), _p(by), _p(bz), _p(phi), _p(rhs_), _p(out))
    return out


def rbgs_color(g, bx, by, bz, rhs_, phi, color):
    lib().orc_rbgs_color(C.byref(g), _p(bx), _p(by), _p(bz), _p(rhs_), _p(phi), int(color))


def rbgs_sweep(g, bx, by, bz, rhs_, phi):
    lib().orc_rbgs_sweep(C.byref(g), _p(bx), _p(by), _p(bz), _p(rhs_), _p(phi))


def can_coarsen(g, coarsest_n=4) -> bool:
    return bool(lib().orc_can_coarsen(C.byref(g), coarsest_n))


def coarsen_coeff(g, bx, by, bz):
    c = coarsen_grid(g)
    cbx, cby, cbz = (np.empty(face_shape(c, d)) for d in range(3))
    lib().orc_coarsen_coeff(C.byref(g), _p(bx), _p(by), _p(bz), _p(cbx), _p(cby), _p(cbz))
    return c, cbx, cby, cbz


def restrict(g, fine):
    c = coarsen_grid(g)
    out = np.empty(cell_shape(c))
    lib().orc_restrict(C.byref(g), _p(fine), _p(out))
    return out


def prolong_add(g, coarse, fine, prolongation=0):
    lib().orc_prolong_add(C.byref(g), _p(coarse), _p(fine), int(prolongation))


def bottom_solve(g, bx, by, bz, f):
    e = np.zeros(cell_shape(g))
    st = lib().orc_bottom_solve(C.byref(g), _p(bx), _p(by), _p(bz), _p(f), _p(e))
    if st != 0:
        raise RuntimeError("orc_bottom_solve failed")
    return e


def vcycle(g, bx, by, bz, rhs_, phi, mg):
    return lib().orc_vcycle(C.byref(g), _p(bx), _p(by), _p(bz), _p(rhs_), _p(phi), C.byref(mg))


def correct(g, rho, phi, u, v, w):
    lib().orc_correct(C.byref(g), _p(rho), _p(phi), _p(u), _p(v), _p(w))


def project(g, b, mg, beta0, rho0, rho, u, v, w, S=None, want_phi=True):
    """Runs O9.  u, v, w are corrected IN PLACE.  Returns (status, phi, stats-dict)."""
    phi = np.zeros(cell_shape(g)) if want_phi else None
    st = Stats()
    status = lib().orc_project(C.byref(g), C.byref(b), C.byref(mg), _p(beta0), _p(rho0), _p(rho),
                               _p(u), _p(v), _p(w), _p(S), _p(phi), C.byref(st))
    stats = dict(cycles=st.cycles, singular=st.singular, levels=st.levels,
                 converged=st.converged, rhs_norm_inf=st.rhs_norm_inf,
                 res_norm_inf=st.res_norm_inf, rhs_mean_removed=st.rhs_mean_removed,
                 res_history=list(st.res_history[:min(st.cycles, 128)]))
    return status, phi, stats


def num_threads() -> int:
    return lib().orc_num_threads()


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))
