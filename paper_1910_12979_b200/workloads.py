"""Seeded synthetic input generators for the MAC projection (numpy only).

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench) and therefore
holds none of the method's arithmetic: no operator, no smoother, no multigrid.  It only builds the
inputs named by BASELINE.json's five configs, with the readings of SURVEY.md Sec. 8(d) / DESIGN.md
"Input recipe".  They stand in for the paper's `reacting_bubble` runs, whose setup
files are not available: a 1-D stratified base state under a 3-D perturbed density,
planar and spherical geometry, heating concentrated where burning occurs.

Array shapes are numpy C order with x fastest: cells [nz, ny, nx]; u [nz, ny, nx+1];
v [nz, ny+1, nx]; w [nz+1, ny, nx].  Random draws use numpy.random.Generator(PCG64(seed)) in the
fixed order documented per config (rho-noise, velocity fields, S parameters).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from functools import lru_cache

import numpy as np

PERIODIC, WALL, OUTFLOW = 0, 1, 2
PLANAR, SPHERICAL = 0, 1


@dataclass
class Workload:
    name: str
    n: tuple                      # (nx, ny, nz)
    dx: tuple                     # (dx, dy, dz)
    bc_lo: tuple
    bc_hi: tuple
    geometry: int
    nr: int
    dr: float
    center: tuple
    beta0: np.ndarray             # [nr]
    rho0: np.ndarray              # [nr]
    rho: np.ndarray               # [nz, ny, nx]
    u: np.ndarray
    v: np.ndarray
    w: np.ndarray
    S: np.ndarray | None
    rel_tol: float = 1e-10
    nu_pre: int = 2
    nu_post: int = 2
    max_cycles: int = 100
    seed: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def ncells(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]


# ------------------------------------------------------------------------------------------------
# Lane-Emden (textbook polytrope):  theta'' + (2/xi) theta' + theta^n = 0, theta(0)=1, theta'(0)=0
# ------------------------------------------------------------------------------------------------

@lru_cache(maxsize=8)
def lane_emden(n: float, dxi: float = 1e-4):
    """RK4 from the series start theta = 1 - xi^2/6 + n xi^4/120.  Returns (xi, theta, dtheta)
    up to and including the first step with theta <= 0."""
    def f(xi, y, z):
        return z, -(max(y, 0.0) ** n) - 2.0 * z / xi

    xi = dxi
    y = 1.0 - xi * xi / 6.0 + n * xi ** 4 / 120.0
    z = -xi / 3.0 + n * xi ** 3 / 30.0
    xs, ys, zs = [0.0, xi], [1.0, y], [0.0, z]
    while y > 0.0 and xi < 20.0:
        k1y, k1z = f(xi, y, z)
        k2y, k2z = f(xi + 0.5 * dxi, y + 0.5 * dxi * k1y, z + 0.5 * dxi * k1z)
        k3y, k3z = f(xi + 0.5 * dxi, y + 0.5 * dxi * k2y, z + 0.5 * dxi * k2z)
        k4y, k4z = f(xi + dxi, y + dxi * k3y, z + dxi * k3z)
        y += dxi * (k1y + 2 * k2y + 2 * k3y + k4y) / 6.0
        z += dxi * (k1z + 2 * k2z + 2 * k3z + k4z) / 6.0
        xi += dxi
        xs.append(xi)
        ys.append(y)
        zs.append(z)
    return np.array(xs), np.array(ys), np.array(zs)


def lane_emden_first_zero(n: float):
    """(xi_1, -xi_1^2 theta'(xi_1)) by linear interpolation across the sign change."""
    xs, ys, zs = lane_emden(n)
    a, b = len(xs) - 2, len(xs) - 1
    t = ys[a] / (ys[a] - ys[b])
    xi1 = xs[a] + t * (xs[b] - xs[a])
    dth = zs[a] + t * (zs[b] - zs[a])
    return xi1, -xi1 * xi1 * dth


# ------------------------------------------------------------------------------------------------
# helpers (coordinates, profile sampling for INPUT construction only)
# ------------------------------------------------------------------------------------------------

def _centres(n, h):
    return (np.arange(n) + 0.5) * h


def _profile_r(nr, dr):
    return (np.arange(nr) + 0.5) * dr


def _interp_profile(f, dr, r):
    """Input-side sampling of a radial profile (np.interp holds the end values constant)."""
    return np.interp(r, _profile_r(len(f), dr), f)


def _gaussian_bumps(rng, N, nb=8, periodic_xy=True):
    """S = sum of nb Gaussian bumps; draws: centres (nb x 3), widths (nb), amplitudes (nb)."""
    ctr = rng.uniform(0.0, 1.0, size=(nb, 3))
    wid = rng.uniform(0.05, 0.15, size=nb)
    amp = rng.uniform(0.5, 1.5, size=nb)
    c = _centres(N, 1.0 / N)
    S = np.zeros((N, N, N))
    for b in range(nb):
        ddx = np.abs(c - ctr[b, 0])
        ddy = np.abs(c - ctr[b, 1])
        if periodic_xy:
            ddx = np.minimum(ddx, 1.0 - ddx)
            ddy = np.minimum(ddy, 1.0 - ddy)
        ddz = c - ctr[b, 2]
        gx = np.exp(-0.5 * (ddx / wid[b]) ** 2)
        gy = np.exp(-0.5 * (ddy / wid[b]) ** 2)
        gz = np.exp(-0.5 * (ddz / wid[b]) ** 2)
        S += amp[b] * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    return S


def _close_faces(u, v, w, bc_lo, bc_hi):
    """WALL faces get zero normal velocity; periodic axes: face n := face 0."""
    arr = (u, v, w)
    for d in range(3):
        a = arr[d]
        ax = 2 - d  # numpy axis of direction d
        lo = [slice(None)] * 3
        hi = [slice(None)] * 3
        lo[ax] = 0
        hi[ax] = a.shape[ax] - 1
        if bc_lo[d] == PERIODIC:
            a[tuple(hi)] = a[tuple(lo)]
        else:
            if bc_lo[d] == WALL:
                a[tuple(lo)] = 0.0
            if bc_hi[d] == WALL:
                a[tuple(hi)] = 0.0


# ------------------------------------------------------------------------------------------------
# config 1: triply periodic, beta0 = 1, smooth density, uniform random faces
# ------------------------------------------------------------------------------------------------

def config1(N: int = 32, seed: int = 1000) -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    h = 1.0 / N
    c = _centres(N, h)
    s = np.sin(2 * np.pi * c)
    rho = 1.0 + 0.5 * s[:, None, None] * s[None, :, None] * s[None, None, :]
    u = rng.uniform(-1, 1, size=(N, N, N + 1))
    v = rng.uniform(-1, 1, size=(N, N + 1, N))
    w = rng.uniform(-1, 1, size=(N + 1, N, N))
    bc = (PERIODIC,) * 3
    _close_faces(u, v, w, bc, bc)
    return Workload("config1_periodic", (N, N, N), (h, h, h), bc, bc, PLANAR, N, h, (0, 0, 0),
                    np.ones(N), np.ones(N), rho, u, v, w, None, seed=seed)


# ------------------------------------------------------------------------------------------------
# configs 2 and 5: plane-parallel atmospheres, periodic x/y, walls in z
# ------------------------------------------------------------------------------------------------

def _planar(name, N, seed, rho0, beta0, vel_seed=None):
    rng = np.random.Generator(np.random.PCG64(seed))
    h = 1.0 / N
    rho = rho0[:, None, None] * (1.0 + 1e-2 * rng.standard_normal((N, N, N)))
    vr = rng if vel_seed is None else np.random.Generator(np.random.PCG64(vel_seed))
    u = 0.1 * vr.standard_normal((N, N, N + 1))
    v = 0.1 * vr.standard_normal((N, N + 1, N))
    w = 0.1 * vr.standard_normal((N + 1, N, N))
    S = _gaussian_bumps(rng, N)
    # reading A23: zero beta0-weighted mean so that D(beta0 U) = beta0 S is reachable between walls
    S -= (beta0[:, None, None] * S).sum() / (beta0.sum() * N * N)
    bc_lo = (PERIODIC, PERIODIC, WALL)
    bc_hi = (PERIODIC, PERIODIC, WALL)
    _close_faces(u, v, w, bc_lo, bc_hi)
    return Workload(name, (N, N, N), (h, h, h), bc_lo, bc_hi, PLANAR, N, h, (0, 0, 0),
                    beta0, rho0, rho, u, v, w, S, seed=seed)


def config2(N: int = 128, seed: int = 2000) -> Workload:
    z = _centres(N, 1.0 / N)
    rho0 = np.exp(-z / 0.2)
    return _planar("config2_planar_atmosphere", N, seed, rho0, rho0 ** 0.6)


def config5(N: int = 1024, seed: int = 5000, step: int = 0) -> Workload:
    """n = 3 plane-parallel polytrope (reading A21).  rho and S come from `seed`; the face
    velocities are redrawn per step from seed + 1 + step."""
    z = _centres(N, 1.0 / N)
    theta = 1.0 - 0.9 * z
    wl = _planar("config5_convective_shell", N, seed, theta ** 3, theta ** 2.4,
                 vel_seed=seed + 1 + step)
    wl.meta["step"] = step
    return wl


# ------------------------------------------------------------------------------------------------
# configs 3 and 4: spherical star in a box
# ------------------------------------------------------------------------------------------------

def star_profile(N: int, contrast: float, beta_exponent: float = 0.6):
    """n = 1.5 Lane-Emden density scaled so rho0(r = 1/2) = 1/contrast, floor beyond (A20, A22).
    Returns (nr, dr, rho0[nr], beta0[nr])."""
    h = 1.0 / N
    dr = 0.5 * h
    nr = int(math.ceil(0.5 * math.sqrt(3.0) / dr)) + 1
    xs, th, _ = lane_emden(1.5)
    theta_edge = (1.0 / contrast) ** (1.0 / 1.5)
    # theta is monotonically decreasing: invert by interpolation on the reversed arrays
    xi_edge = float(np.interp(theta_edge, th[::-1], xs[::-1]))
    alpha = 0.5 / xi_edge
    r = _profile_r(nr, dr)
    theta_r = np.interp(r / alpha, xs, th)
    rho0 = np.where(r < 0.5, np.maximum(theta_r, 0.0) ** 1.5, 1.0 / contrast)
    rho0 = np.maximum(rho0, 1.0 / contrast)
    return nr, dr, rho0, rho0 ** beta_exponent


def _star(name, N, seed, contrast, bc_kind, beta_exponent=0.6):
    rng = np.random.Generator(np.random.PCG64(seed))
    h = 1.0 / N
    nr, dr, rho0, beta0 = star_profile(N, contrast, beta_exponent)
    c = _centres(N, h) - 0.5
    f = np.arange(N + 1) * h - 0.5
    r_cell = np.sqrt(c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2)
    rho = _interp_profile(rho0, dr, r_cell) * (1.0 + 1e-3 * rng.standard_normal((N, N, N)))
    S = np.where(r_cell < 0.15, np.cos(np.pi * r_cell / (2 * 0.15)) ** 2, 0.0)
    del r_cell
    # solenoidal part: discrete curl of an edge-centred vector potential, divided by beta0 on the
    # face so that D(beta0 U_sol) = 0 (up to how the path samples beta0 on faces)
    Ax = rng.uniform(-1, 1, size=(N + 1, N + 1, N))
    Ay = rng.uniform(-1, 1, size=(N + 1, N, N + 1))
    Az = rng.uniform(-1, 1, size=(N, N + 1, N + 1))
    Fx = np.diff(Az, axis=1) / h - np.diff(Ay, axis=0) / h
    Fy = np.diff(Ax, axis=0) / h - np.diff(Az, axis=2) / h
    Fz = np.diff(Ay, axis=2) / h - np.diff(Ax, axis=1) / h
    del Ax, Ay, Az
    rms = math.sqrt((np.sum(Fx ** 2) + np.sum(Fy ** 2) + np.sum(Fz ** 2)) / (Fx.size + Fy.size + Fz.size))
    bfx = _interp_profile(beta0, dr, np.sqrt(c[:, None, None] ** 2 + c[None, :, None] ** 2 + f[None, None, :] ** 2))
    u = Fx / (rms * bfx) + 1e-2 * rng.standard_normal(Fx.shape)
    del Fx, bfx
    bfy = _interp_profile(beta0, dr, np.sqrt(c[:, None, None] ** 2 + f[None, :, None] ** 2 + c[None, None, :] ** 2))
    v = Fy / (rms * bfy) + 1e-2 * rng.standard_normal(Fy.shape)
    del Fy, bfy
    bfz = _interp_profile(beta0, dr, np.sqrt(f[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2))
    w = Fz / (rms * bfz) + 1e-2 * rng.standard_normal(Fz.shape)
    del Fz, bfz
    bc = (bc_kind,) * 3
    _close_faces(u, v, w, bc, bc)
    wl = Workload(name, (N, N, N), (h, h, h), bc, bc, SPHERICAL, nr, dr, (0.5, 0.5, 0.5),
                  beta0, rho0, rho, u, v, w, S, seed=seed)
    wl.meta.update(contrast=contrast, beta_exponent=beta_exponent)
    return wl


def config3(N: int = 256, seed: int = 3000, variant: str = "N", beta_exponent: float = 0.6) -> Workload:
    """variant 'N': WALL on all six sides (singular, mean removed); 'D': OUTFLOW on all sides (A9)."""
    return _star(f"config3{variant}_star_1e4", N, seed, 1e4, WALL if variant == "N" else OUTFLOW, beta_exponent)


def config4(N: int = 512, seed: int = 4000, variant: str = "N", beta_exponent: float = 0.6) -> Workload:
    return _star(f"config4{variant}_star_1e6", N, seed, 1e6, WALL if variant == "N" else OUTFLOW, beta_exponent)


def by_name(name: str, N: int | None = None, seed: int | None = None) -> Workload:
    """'1', '2', '3N', '3D', '4N', '4D', '5' (optionally with a reduced N)."""
    table = {"1": (config1, {}), "2": (config2, {}), "3N": (config3, {"variant": "N"}),
             "3D": (config3, {"variant": "D"}), "4N": (config4, {"variant": "N"}),
             "4D": (config4, {"variant": "D"}), "5": (config5, {})}
    fn, kw = table[name]
    kw = dict(kw)
    if N is not None:
        kw["N"] = N
    if seed is not None:
        kw["seed"] = seed
    return fn(**kw)


def with_base_state(wl: Workload, gamma: float = 5.0 / 3.0, seed: int = 77) -> Workload:
    """Adds the 1-D thermodynamic base state that Eq. 5 / Eq. 6 of the paper consume to a
    workload, in wl.meta: p0 = rho0^gamma (a polytrope consistent with the density profile), Gamma1bar = gamma
    (1 + 2 % smooth variation) and a smooth dp0/dt of a few per cent of p0 per unit time.  Inputs only."""
    rng = np.random.Generator(np.random.PCG64(seed))
    r = _profile_r(wl.nr, wl.dr)
    L = r[-1] + 0.5 * wl.dr
    ph = rng.uniform(0.0, 2.0 * np.pi, size=2)
    wl.meta["p0"] = wl.rho0 ** gamma
    wl.meta["gamma1bar"] = gamma * (1.0 + 0.02 * np.sin(2.0 * np.pi * r / L + ph[0]))
    wl.meta["dp0dt"] = 0.05 * wl.meta["p0"] * np.cos(3.0 * np.pi * r / L + ph[1])
    return wl


def mixed_bc_case(n=(16, 8, 12), seed: int = 7, bc_lo=(OUTFLOW, WALL, PERIODIC),
                  bc_hi=(WALL, OUTFLOW, PERIODIC), geometry: int = PLANAR) -> Workload:
    """Small non-cubic case with every boundary type and anisotropic spacing (edge-case tests)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nx, ny, nz = n
    dx = (1.0 / nx, 0.8 / ny, 1.3 / nz)
    if geometry == PLANAR:
        nr, dr, center = nz, dx[2], (0.0, 0.0, 0.0)
    else:
        dr = 0.5 * min(dx)
        nr = int(math.ceil(math.sqrt(1.0 + 0.64 + 1.69) / dr)) + 1
        center = (0.45, 0.4, 0.6)
    r = _profile_r(nr, dr)
    rho0 = np.exp(-r / 0.4)
    beta0 = rho0 ** 0.6
    rho = np.exp(rng.uniform(-1.0, 1.0, size=(nz, ny, nx)))
    u = rng.uniform(-1, 1, size=(nz, ny, nx + 1))
    v = rng.uniform(-1, 1, size=(nz, ny + 1, nx))
    w = rng.uniform(-1, 1, size=(nz + 1, ny, nx))
    S = rng.uniform(-1, 1, size=(nz, ny, nx))
    _close_faces(u, v, w, bc_lo, bc_hi)
    return Workload("mixed_bc", tuple(n), dx, tuple(bc_lo), tuple(bc_hi), geometry, nr, dr, center,
                    beta0, rho0, rho, u, v, w, S, seed=seed)


def cell_centred(wl: Workload):
    """Cell-centred velocities for the end-of-step (nodal) projection from a workload's face velocities: the mean of
    the two faces of a cell per axis (input construction only).  Returns (uc, vc, wc), each [nz, ny, nx]."""
    uc = np.ascontiguousarray(0.5 * (wl.u[:, :, :-1] + wl.u[:, :, 1:]))
    vc = np.ascontiguousarray(0.5 * (wl.v[:, :-1, :] + wl.v[:, 1:, :]))
    wc = np.ascontiguousarray(0.5 * (wl.w[:-1, :, :] + wl.w[1:, :, :]))
    return uc, vc, wc
