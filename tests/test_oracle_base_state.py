"""Pins of the oracle's base-state steps O11 / O12 (Eq. 5, Eq. 6): closed forms,
convergence order against an analytic integral, brute force per cell.  CPU only."""
import numpy as np
import pytest

from helpers import oracle_structs
from paper_1910_12979_b200 import workloads as W


def samples(nr, L=1.0):
    dr = L / nr
    return (np.arange(nr) + 0.5) * dr, dr


def test_P14_beta0_closed_form_constant_gamma(oracle):
    """Eq. 5 with constant Gamma1bar integrates exactly: beta0 = rho0(0) (p0 / p0(0))^(1/Gamma1bar); for a polytrope
    p0 = K rho0^Gamma with Gamma = Gamma1bar that is beta0 = rho0 (the isentropic atmosphere)."""
    r, _ = samples(200)
    rho0 = (1.0 - 0.9 * r) ** 3
    for gam in (5.0 / 3.0, 4.0 / 3.0, 1.1):
        p0 = 2.5 * rho0 ** gam
        b = oracle.make_beta0(rho0, p0, np.full_like(r, gam))
        assert np.abs(b / rho0 - 1.0).max() <= 1e-13
        p0 = np.exp(-r / 0.2)                    # isothermal-like pressure, same Gamma1bar
        b = oracle.make_beta0(rho0, p0, np.full_like(r, gam))
        assert np.abs(b / (rho0[0] * (p0 / p0[0]) ** (1.0 / gam)) - 1.0).max() <= 1e-13


def test_P15_beta0_second_order_for_varying_gamma(oracle):
    """Gamma1bar = a + b r, p0 = exp(-r/H): ln(beta0 / beta0(r_0)) = -(1/(b H)) ln((a + b r)/(a + b r_0)).
    The midpoint rule in ln p0 is second order: the error drops by 4 when nr doubles."""
    a, bb, H = 1.4, 0.5, 0.2
    errs = []
    for nr in (32, 64, 128, 256):
        r, _ = samples(nr)
        p0 = np.exp(-r / H)
        rho0 = np.full_like(r, 3.0)
        got = oracle.make_beta0(rho0, p0, a + bb * r)
        exact = rho0[0] * ((a + bb * r) / (a + bb * r[0])) ** (-1.0 / (bb * H))
        errs.append(np.abs(got / exact - 1.0).max())
    ratios = [errs[q] / errs[q + 1] for q in range(3)]
    assert errs[-1] < 2e-6 and all(3.6 < x < 4.4 for x in ratios), (errs, ratios)


def test_P16_dpdt_term_and_effective_source_brute_force(oracle):
    """q = dp0dt / (Gamma1bar p0) sample by sample; S_eff = S - q(r_cell), per-cell loop in spherical geometry."""
    wl = W.mixed_bc_case(n=(6, 5, 7), geometry=W.SPHERICAL, seed=3)
    g, b, _ = oracle_structs(oracle, wl)
    rng = np.random.default_rng(5)
    p0 = np.exp(rng.uniform(-1, 1, wl.nr)); gam = rng.uniform(1.2, 1.7, wl.nr); dpdt = rng.uniform(-1, 1, wl.nr)
    q = oracle.dpdt_term(p0, gam, dpdt)
    assert np.array_equal(q, np.array([dpdt[m] / (gam[m] * p0[m]) for m in range(wl.nr)]))
    got = oracle.effective_source(g, b, wl.S, q)
    nx, ny, nz = wl.n
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                x, y, z = (i + 0.5) * wl.dx[0], (j + 0.5) * wl.dx[1], (k + 0.5) * wl.dx[2]
                rr = np.sqrt((x - wl.center[0]) ** 2 + (y - wl.center[1]) ** 2 + (z - wl.center[2]) ** 2)
                s = rr / wl.dr - 0.5                         # O1 written out: linear between samples, constant beyond
                if s <= 0: qq = q[0]
                elif s >= wl.nr - 1: qq = q[-1]
                else:
                    m = int(s); t = s - m; qq = (1 - t) * q[m] + t * q[m + 1]
                assert got[k, j, i] == pytest.approx(wl.S[k, j, i] - qq, rel=1e-13, abs=1e-15)
    # S = NULL means 0
    assert np.array_equal(oracle.effective_source(g, b, None, q), -oracle.rho_from_profile(g, b, q))


def test_P17_constraint_of_eq6_holds_with_the_dpdt_term(oracle):
    """Projecting with S_eff enforces D(beta0 U) = beta0 (S - (1/(Gamma1bar p0)) dp0/dt) (Eq. 6) to rel_tol."""
    wl = W.with_base_state(W.config3(N=16, variant="D"))
    g, b, mg = oracle_structs(oracle, wl)
    beta0 = oracle.make_beta0(wl.rho0, wl.meta["p0"], wl.meta["gamma1bar"])
    q = oracle.dpdt_term(wl.meta["p0"], wl.meta["gamma1bar"], wl.meta["dp0dt"])
    S_eff = oracle.effective_source(g, b, wl.S, q)
    u, v, w = wl.u.copy(), wl.v.copy(), wl.w.copy()
    st, phi, stats = oracle.project(g, b, mg, beta0, wl.rho0, wl.rho, u, v, w, S_eff)
    assert st == 0
    c = oracle.constraint(g, b, beta0, u, v, w, wl.S) + oracle.rho_from_profile(g, b, beta0) * oracle.rho_from_profile(g, b, q)
    assert np.abs(c).max() <= wl.rel_tol * stats["rhs_norm_inf"] * 1.01
