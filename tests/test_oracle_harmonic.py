"""Pins of the harmonic face-density variant (reading A3: the face takes the mean of 1/rho instead of the mean of
rho; oracle flag orc_grid.rho_mean = 1).  CPU only."""
import numpy as np
import pytest

from helpers import oracle_project, oracle_structs, rel_l2
from paper_1910_12979_b200 import workloads as W

PER, WALL, OUT = W.PERIODIC, W.WALL, W.OUTFLOW


def harmonic(wl):
    wl.meta["rho_mean"] = 1
    return wl


def test_face_coeff_harmonic_brute_force(oracle):
    """b = beta0(face) * (1/rho_L + 1/rho_R)/2 on every face, per-face loop (planar, mixed boundaries)."""
    wl = harmonic(W.mixed_bc_case(n=(6, 5, 7), bc_lo=(OUT, WALL, PER), bc_hi=(WALL, OUT, PER)))
    g, b, _ = oracle_structs(oracle, wl)
    bx, by, bz = oracle.face_coeff(g, b, wl.beta0, wl.rho)
    nx, ny, nz = wl.n
    rho = wl.rho
    for k in range(nz):
        for j in range(ny):
            for i in range(nx + 1):                     # x faces: OUTFLOW low, WALL high -> one interior cell at the ends
                lo, hi = (0, 0) if i == 0 else ((nx - 1, nx - 1) if i == nx else (i - 1, i))
                inv = 0.5 * (1.0 / rho[k, j, lo] + 1.0 / rho[k, j, hi])
                assert bx[k, j, i] == pytest.approx(wl.beta0[k] * inv, rel=1e-14)
    for k in range(nz + 1):                             # z faces: periodic wrap, beta0 of the face (A18: position 0 at the seam)
        lo, hi = (nz - 1, 0) if k in (0, nz) else (k - 1, k)
        bf = wl.beta0[0] if k in (0, nz) else 0.5 * (wl.beta0[k - 1] + wl.beta0[k])
        inv = 0.5 * (1.0 / rho[lo, 2, 3] + 1.0 / rho[hi, 2, 3])
        assert bz[k, 2, 3] == pytest.approx(bf * inv, rel=1e-14)


def test_harmonic_equals_arithmetic_where_rho_is_uniform(oracle):
    wl = W.config1(N=8)
    wl.rho[:] = 1.7
    a = oracle_project(oracle, wl)
    h = oracle_project(oracle, harmonic(wl))
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(h[key], a[key]) <= 1e-13


@pytest.mark.parametrize("name,N", [("2", 16), ("3D", 16), ("mixed", 0)])
def test_harmonic_constraint_identity_and_difference(oracle, name, N):
    """P4/P5 with the harmonic face density: the coefficient (O3) and the correction (O10) use the same rho_face, so
    D(beta0 U_new) - beta0 S - m == rhs - L phi holds to rounding and the constraint to rel_tol; and the variant is
    really a different discretisation (the result moves)."""
    wl = W.mixed_bc_case(n=(16, 8, 12)) if name == "mixed" else W.by_name(name, N)
    a = oracle_project(oracle, wl)
    h = oracle_project(oracle, harmonic(wl))
    assert h["status"] == 0
    O, g, b = oracle, h["g"], h["b"]
    bf = O.face_coeff(g, b, wl.beta0, wl.rho)
    rhs = O.rhs(g, b, wl.beta0, wl.u, wl.v, wl.w, wl.S)
    m = h["stats"]["rhs_mean_removed"]
    res = O.residual(g, *bf, h["phi"], rhs - m)
    c = O.constraint(g, b, wl.beta0, h["u"], h["v"], h["w"], wl.S) - m
    assert np.abs(c - res).max() <= 1e-13 * np.abs(rhs).max()
    assert np.abs(c).max() <= wl.rel_tol * h["stats"]["rhs_norm_inf"] * 1.01
    assert rel_l2(h["u"], a["u"]) > 1e-6
