"""Shared test helpers: workload -> oracle structs, norms.  No method arithmetic."""
import numpy as np


def oracle_structs(O, wl, **mg_kw):
    g = O.make_grid(wl.n, wl.dx, wl.bc_lo, wl.bc_hi, rho_mean=wl.meta.get("rho_mean", 0))
    b = O.make_base(wl.geometry, wl.nr, wl.dr, wl.center)
    kw = dict(nu_pre=wl.nu_pre, nu_post=wl.nu_post, max_cycles=wl.max_cycles, rel_tol=wl.rel_tol)
    kw.update(mg_kw)
    return g, b, O.make_mg(**kw)


def oracle_project(O, wl, **mg_kw):
    """Run the oracle on copies of the workload's velocities.  Returns dict."""
    g, b, mg = oracle_structs(O, wl, **mg_kw)
    u, v, w = wl.u.copy(), wl.v.copy(), wl.w.copy()
    status, phi, stats = O.project(g, b, mg, wl.beta0, wl.rho0, wl.rho, u, v, w, wl.S)
    return dict(status=status, phi=phi, u=u, v=v, w=w, stats=stats, g=g, b=b, mg=mg)


def rel_l2(a, b):
    d = np.linalg.norm((a - b).ravel())
    n = np.linalg.norm(b.ravel())
    return d / n if n > 0 else d
