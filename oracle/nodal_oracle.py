"""ctypes loader for the nodal-projection ORACLE (oracle/nodal_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
All arithmetic is in nodal_oracle.c (readings N1..N10 in nodal_oracle.h); this file only marshals numpy arrays.
Grid / Base / MG / Stats and make_* come from the MAC oracle's loader (same grid, same base state).

Shapes (numpy C order, x fastest): cells [nz, ny, nx]; nodes [nz+1, ny+1, nx+1]; u, v, w are CELL arrays here.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import mac_oracle as M
from .mac_oracle import Grid, Base, MG, Stats, make_grid, make_base, make_mg, cell_shape, _p, _DP  # noqa: F401

_bound = False


def lib():
    global _bound
    L = M.lib()
    if not _bound:
        GP, BP, MP = C.POINTER(Grid), C.POINTER(Base), C.POINTER(MG)
        L.nod_omega.restype = C.c_double
        L.nod_omega.argtypes = [GP]
        L.nod_node_kind.argtypes = [GP, C.POINTER(C.c_int)]
        L.nod_weights.argtypes = [GP, _DP]
        L.nod_sigma.argtypes = [GP, BP, _DP, _DP, _DP]
        L.nod_apply.argtypes = [GP, _DP, _DP, _DP]
        L.nod_diag.argtypes = [GP, _DP, _DP]
        L.nod_residual.argtypes = [GP, _DP, _DP, _DP, _DP]
        L.nod_rhs.argtypes = [GP, BP, _DP, _DP, _DP, _DP, _DP, _DP]
        L.nod_constraint.argtypes = [GP, BP, _DP, _DP, _DP, _DP, _DP, _DP]
        L.nod_jacobi.argtypes = [GP, _DP, _DP, _DP, C.c_double]
        L.nod_coarsen_sigma.argtypes = [GP, _DP, _DP]
        L.nod_restrict.argtypes = [GP, _DP, _DP]
        L.nod_prolong_add.argtypes = [GP, _DP, _DP]
        L.nod_bottom_solve.restype = C.c_int
        L.nod_bottom_solve.argtypes = [GP, _DP, _DP, _DP]
        L.nod_vcycle.restype = C.c_int
        L.nod_vcycle.argtypes = [GP, _DP, _DP, _DP, MP]
        L.nod_correct.argtypes = [GP, _DP, _DP, _DP, _DP, _DP]
        L.nod_weighted_mean.restype = C.c_double
        L.nod_weighted_mean.argtypes = [GP, _DP]
        L.nod_norm_inf.restype = C.c_double
        L.nod_norm_inf.argtypes = [GP, _DP]
        L.nod_project.restype = C.c_int
        L.nod_project.argtypes = [GP, BP, MP, _DP, _DP, _DP, _DP, _DP, _DP, _DP, _DP, C.POINTER(Stats)]
        _bound = True
    return L


def node_shape(g: Grid):
    return (g.n[2] + 1, g.n[1] + 1, g.n[0] + 1)


def omega(g) -> float:
    return lib().nod_omega(C.byref(g))


def node_kind(g):
    out = np.zeros(node_shape(g), dtype=np.int32)
    lib().nod_node_kind(C.byref(g), out.ctypes.data_as(C.POINTER(C.c_int)))
    return out


def weights(g):
    out = np.empty(node_shape(g))
    lib().nod_weights(C.byref(g), _p(out))
    return out


def sigma(g, b, beta0, rho):
    out = np.empty(cell_shape(g))
    lib().nod_sigma(C.byref(g), C.byref(b), _p(beta0), _p(rho), _p(out))
    return out


def apply(g, sig, phi):
    out = np.empty(node_shape(g))
    lib().nod_apply(C.byref(g), _p(sig), _p(phi), _p(out))
    return out


def diag(g, sig):
    out = np.empty(node_shape(g))
    lib().nod_diag(C.byref(g), _p(sig), _p(out))
    return out


def residual(g, sig, phi, rhs_):
    out = np.empty(node_shape(g))
    lib().nod_residual(C.byref(g), _p(sig), _p(phi), _p(rhs_), _p(out))
    return out


def rhs(g, b, beta0, u, v, w, S=None):
    out = np.empty(node_shape(g))
    lib().nod_rhs(C.byref(g), C.byref(b), _p(beta0), _p(u), _p(v), _p(w), _p(S), _p(out))
    return out


def constraint(g, b, beta0, u, v, w, S=None):
    out = np.empty(node_shape(g))
    lib().nod_constraint(C.byref(g), C.byref(b), _p(beta0), _p(u), _p(v), _p(w), _p(S), _p(out))
    return out


def jacobi(g, sig, rhs_, phi, om=None):
    lib().nod_jacobi(C.byref(g), _p(sig), _p(rhs_), _p(phi), float(omega(g) if om is None else om))


def coarsen_sigma(g, sig):
    c = M.coarsen_grid(g)
    out = np.empty(cell_shape(c))
    lib().nod_coarsen_sigma(C.byref(g), _p(sig), _p(out))
    return c, out


def restrict(g, fine):
    c = M.coarsen_grid(g)
    out = np.empty(node_shape(c))
    lib().nod_restrict(C.byref(g), _p(fine), _p(out))
    return out


def prolong_add(g, coarse, fine):
    lib().nod_prolong_add(C.byref(g), _p(coarse), _p(fine))


def bottom_solve(g, sig, f):
    e = np.zeros(node_shape(g))
    if lib().nod_bottom_solve(C.byref(g), _p(sig), _p(f), _p(e)) != 0:
        raise RuntimeError("nod_bottom_solve failed")
    return e


def vcycle(g, sig, rhs_, phi, mg):
    return lib().nod_vcycle(C.byref(g), _p(sig), _p(rhs_), _p(phi), C.byref(mg))


def correct(g, rho, phi, u, v, w):
    lib().nod_correct(C.byref(g), _p(rho), _p(phi), _p(u), _p(v), _p(w))


def weighted_mean(g, f) -> float:
    return lib().nod_weighted_mean(C.byref(g), _p(f))


def norm_inf(g, f) -> float:
    return lib().nod_norm_inf(C.byref(g), _p(f))


def project(g, b, mg, beta0, rho0, rho, u, v, w, S=None, want_phi=True):
    """The whole nodal projection.  u, v, w (cell arrays) are corrected IN PLACE.  Returns (status, phi, stats)."""
    phi = np.zeros(node_shape(g)) if want_phi else None
    st = Stats()
    status = lib().nod_project(C.byref(g), C.byref(b), C.byref(mg), _p(beta0), _p(rho0), _p(rho), _p(u), _p(v), _p(w),
                               _p(S), _p(phi), C.byref(st))
    stats = dict(cycles=st.cycles, singular=st.singular, levels=st.levels, converged=st.converged,
                 rhs_norm_inf=st.rhs_norm_inf, res_norm_inf=st.res_norm_inf, rhs_mean_removed=st.rhs_mean_removed,
                 res_history=list(st.res_history[:min(st.cycles, 128)]))
    return status, phi, stats
