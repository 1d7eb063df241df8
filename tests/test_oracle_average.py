"""Pins of the oracle's lateral average O13 (rho0 is the lateral average of rho).  CPU only."""
import numpy as np
import pytest

from helpers import oracle_structs
from paper_1910_12979_b200 import workloads as W


def test_P18_planar_average_is_the_plane_mean(oracle):
    """Planar, nr = nz, dr = dz: rho0[k] = mean of plane k (numpy's mean over the lateral axes)."""
    wl = W.config2(N=16)
    g, b, _ = oracle_structs(oracle, wl)
    rho0, cnt = oracle.lateral_average(g, b, wl.rho)
    assert np.all(cnt == 16 * 16)
    assert np.allclose(rho0, wl.rho.mean(axis=(1, 2)), rtol=1e-14, atol=0)


def test_P19_spherical_binning_brute_force_and_conservation(oracle):
    """Per-cell Python loop: membership m = min(nr-1, floor(r/dr)), bin means, and the fill of empty samples by
    linear interpolation in m (constant beyond the ends); sum_m count_m rho0_m = sum of rho."""
    wl = W.mixed_bc_case(n=(6, 5, 7), geometry=W.SPHERICAL, seed=4)
    g, b, _ = oracle_structs(oracle, wl)
    rho0, cnt = oracle.lateral_average(g, b, wl.rho)
    nx, ny, nz = wl.n
    sums = np.zeros(wl.nr); c2 = np.zeros(wl.nr, dtype=np.int64)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                x, y, z = (i + 0.5) * wl.dx[0], (j + 0.5) * wl.dx[1], (k + 0.5) * wl.dx[2]
                r = np.sqrt((x - wl.center[0]) ** 2 + (y - wl.center[1]) ** 2 + (z - wl.center[2]) ** 2)
                m = min(wl.nr - 1, int(np.floor(r / wl.dr)))
                sums[m] += wl.rho[k, j, i]; c2[m] += 1
    assert np.array_equal(cnt, c2) and cnt.sum() == nx * ny * nz
    assert (cnt == 0).any()                                    # dr = dx/2: some shells hold no cell centre
    filled = np.nonzero(c2)[0]
    assert np.allclose(rho0[filled], sums[filled] / c2[filled], rtol=1e-14)
    assert np.isclose((rho0[filled] * c2[filled]).sum(), wl.rho.sum(), rtol=1e-13)
    expect = np.interp(np.arange(wl.nr), filled, rho0[filled])   # linear in m, constant beyond the ends
    assert np.allclose(rho0, expect, rtol=1e-14)


def test_P20_average_of_a_radial_field(oracle):
    """A constant field averages to itself in every sample (empty ones included); for rho = f(r) every filled
    sample lies between the extremes of f over its shell."""
    wl = W.config3(N=16, variant="D")
    g, b, _ = oracle_structs(oracle, wl)
    rho0, cnt = oracle.lateral_average(g, b, np.full_like(wl.rho, 2.5))
    assert np.all(rho0 == 2.5)
    field = oracle.rho_from_profile(g, b, wl.rho0)               # rho = rho0(r) exactly, decreasing in r
    avg, cnt = oracle.lateral_average(g, b, field)
    for m in np.nonzero(cnt)[0][:-1]:
        lo, hi = oracle.profile(wl.rho0, wl.dr, (m + 1) * wl.dr), oracle.profile(wl.rho0, wl.dr, m * wl.dr)
        assert lo - 1e-14 <= avg[m] <= hi + 1e-14
