"""GPU-vs-oracle parity of the end-of-step (nodal) projection through the C ABI (maestro_mac_nodal_*).

Per-kernel parity through the step API (bar 1e-13 relative to the array's max-norm over the unknowns), end-to-end
parity with the north_star bar of 1e-10 relative L2 in phi and in the corrected cell velocities, same cycle count.
The oracle is oracle/nodal_oracle.c (readings N1..N10).
"""
import numpy as np
import pytest

from helpers import rel_l2
from paper_1910_12979_b200 import workloads as W

pytestmark = pytest.mark.gpu

PER, WALL, OUT = W.PERIODIC, W.WALL, W.OUTFLOW
KERNEL_TOL = 1e-13
E2E_TOL = 1e-10


@pytest.fixture(scope="module")
def mac():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_12979_b200 import build, mac
    build.build()
    return mac


@pytest.fixture(scope="module")
def N(oracle):
    from oracle import nodal_oracle
    nodal_oracle.lib()
    return nodal_oracle


def tt(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def structs(N, wl, **mg_kw):
    g = N.make_grid(wl.n, wl.dx, wl.bc_lo, wl.bc_hi)
    b = N.make_base(wl.geometry, wl.nr, wl.dr, wl.center)
    kw = dict(nu_pre=wl.nu_pre, nu_post=wl.nu_post, max_cycles=wl.max_cycles, rel_tol=wl.rel_tol)
    kw.update(mg_kw)
    return g, b, N.make_mg(**kw)


def oracle_project(N, wl, **mg_kw):
    g, b, mg = structs(N, wl, **mg_kw)
    u, v, w = W.cell_centred(wl)
    status, phi, st = N.project(g, b, mg, wl.beta0, wl.rho0, wl.rho, u, v, w, wl.S)
    return dict(status=status, phi=phi, u=u, v=v, w=w, stats=st, g=g, b=b)


def gpu_project(mac, wl, **over):
    import torch
    P = mac.MacProjector(mac.desc_from_workload(wl, nodal=1, **over))
    dv = mac.to_device(wl)
    uc, vc, wc = (tt(a) for a in W.cell_centred(wl))
    phi = torch.full((wl.n[2] + 1, wl.n[1] + 1, wl.n[0] + 1), float("nan"), dtype=torch.float64, device="cuda")
    rc, st = P.nodal_project(dv["beta0"], dv["rho0"], dv["rho"], uc, vc, wc, dv["S"], phi)
    out = dict(status=rc, stats=st, phi=phi.cpu().numpy(), u=uc.cpu().numpy(), v=vc.cpu().numpy(), w=wc.cpu().numpy())
    P.close()
    return out


def close(a, b, mask=None, tol=KERNEL_TOL):
    a = a.cpu().numpy() if hasattr(a, "cpu") else a
    if mask is not None:
        a, b = a[mask], b[mask]
    scale = max(np.abs(b).max(), 1e-300)
    return np.abs(a - b).max() <= tol * scale


def small_cases():
    return [
        W.mixed_bc_case(n=(16, 8, 12)),
        W.mixed_bc_case(n=(16, 8, 12), geometry=W.SPHERICAL, seed=11),
        W.mixed_bc_case(n=(24, 20, 8), bc_lo=(PER, WALL, OUT), bc_hi=(PER, WALL, WALL), seed=12),
        W.mixed_bc_case(n=(8, 8, 40), bc_lo=(WALL, PER, PER), bc_hi=(OUT, PER, PER), seed=13),
        W.config1(N=16), W.config2(N=16), W.config3(N=16, variant="N"), W.config3(N=16, variant="D"),
        W.mixed_bc_case(n=(72, 20, 16), bc_lo=(OUT, WALL, PER), bc_hi=(WALL, OUT, PER), seed=14),
        W.mixed_bc_case(n=(136, 28, 16), bc_lo=(WALL, OUT, OUT), bc_hi=(OUT, WALL, WALL), geometry=W.SPHERICAL, seed=15),
        W.mixed_bc_case(n=(64, 24, 16), bc_lo=(PER, PER, WALL), bc_hi=(PER, PER, OUT), seed=16),
    ]


@pytest.mark.parametrize("case", range(11))
def test_nodal_per_kernel_parity(oracle, N, mac, case):
    import torch
    wl = small_cases()[case]
    g, b, mg = structs(N, wl)
    P = mac.MacProjector(mac.desc_from_workload(wl, nodal=1, bottom_rel_tol=1e-13, bottom_max_iter=2000))
    dv = mac.to_device(wl)
    nlev = P.num_levels
    uc, vc, wc = W.cell_centred(wl)

    # sigma on every level
    P.nodal_step_sigma(dv["beta0"], dv["rho0"], dv["rho"])
    sig = N.sigma(g, b, wl.beta0, wl.rho)
    grids, sigs = [g], [sig]
    while oracle.can_coarsen(grids[-1], 4):
        gc, sc = N.coarsen_sigma(grids[-1], sigs[-1])
        grids.append(gc); sigs.append(sc)
    assert nlev == len(grids)
    for l in range(nlev):
        assert close(P.nodal_get(l, mac.NODAL_SIGMA), sigs[l]), l

    # rhs, its max-norm over the unknowns and the removed uniform source
    nrm, mean = P.nodal_step_rhs(tt(uc), tt(vc), tt(wc), dv["S"])
    rhs = N.rhs(g, b, wl.beta0, uc, vc, wc, wl.S)
    kind = N.node_kind(g)
    unk = kind == 0
    m = 0.0
    if oracle.is_singular(g):
        m = rhs[unk].sum() / wl.ncells
        rhs = rhs - m * N.weights(g)
    assert close(P.nodal_get(0, mac.NODAL_RHS), rhs, unk)
    assert nrm == pytest.approx(np.abs(rhs[unk]).max(), rel=1e-12)
    assert mean == pytest.approx(m, abs=1e-13 * np.abs(rhs).max())

    rng = np.random.default_rng(500 + case)
    for l in range(nlev):
        gl, sl = grids[l], sigs[l]
        ul = N.node_kind(gl) == 0
        phi = rng.standard_normal(N.node_shape(gl))
        f = rng.standard_normal(N.node_shape(gl))
        f[~ul] = 0.0
        P.nodal_set(l, mac.NODAL_PHI, tt(phi)); P.nodal_set(l, mac.NODAL_RHS, tt(f))
        assert P.nodal_step_residual_norm(l) == pytest.approx(N.norm_inf(gl, N.residual(gl, sl, phi, f)), rel=1e-12)
        if l + 1 < nlev:
            P.nodal_step_smooth(l, 3)                                  # Jacobi sweeps (ping-pong: odd count)
            ref = phi.copy()
            for _ in range(3):
                N.jacobi(gl, sl, f, ref)
            assert close(P.nodal_get(l, mac.NODAL_PHI), ref, ul), l
            P.nodal_step_residual_restrict(l)
            uc_ = N.node_kind(grids[l + 1]) == 0
            assert close(P.nodal_get(l + 1, mac.NODAL_RHS), N.restrict(gl, N.residual(gl, sl, ref, f)), uc_), l
            assert float(P.nodal_get(l + 1, mac.NODAL_PHI).abs().max()) == 0.0
            ec = rng.standard_normal(N.node_shape(grids[l + 1]))
            P.nodal_set(l + 1, mac.NODAL_PHI, tt(ec))
            P.nodal_step_prolong(l)
            N.prolong_add(gl, ec, ref)
            assert close(P.nodal_get(l, mac.NODAL_PHI), ref, ul), l
        else:
            P.nodal_step_bottom()
            if oracle.is_singular(gl):
                f = f - f[ul].mean() * ul                              # the solvers project f; compare like with like
            e = N.bottom_solve(gl, sl, f)
            assert rel_l2(P.nodal_get(l, mac.NODAL_PHI).cpu().numpy()[ul], e[ul]) <= 1e-9

    # one whole V-cycle from a random state
    phi = rng.standard_normal(N.node_shape(g)); f = rng.standard_normal(N.node_shape(g))
    f[~unk] = 0.0
    if oracle.is_singular(g):
        f[unk] -= f[unk].mean()
    P.nodal_set(0, mac.NODAL_PHI, tt(phi)); P.nodal_set(0, mac.NODAL_RHS, tt(f))
    P.nodal_step_vcycle()
    ref = phi.copy(); N.vcycle(g, sig, f, ref, mg)
    assert rel_l2(P.nodal_get(0, mac.NODAL_PHI).cpu().numpy()[unk], ref[unk]) <= 1e-9

    # correction from a given phi
    P.nodal_set(0, mac.NODAL_PHI, tt(phi))
    u, v, w = tt(uc), tt(vc), tt(wc)
    P.nodal_step_correct(dv["rho0"], dv["rho"], u, v, w)
    ru, rv, rw = uc.copy(), vc.copy(), wc.copy()
    N.correct(g, wl.rho, phi, ru, rv, rw)
    assert close(u, ru) and close(v, rv) and close(w, rw)
    torch.cuda.synchronize()
    P.close()


E2E = [("1", 32), ("2", 32), ("3N", 32), ("3D", 32), ("4N", 32), ("4D", 64), ("5", 32), ("2", 64), ("mixed", 0),
       ("mixed_sph", 0), ("1", 64), ("3N", 128), ("5", 128)]


def get_case(name, n):
    if name == "mixed":
        wl = W.mixed_bc_case(n=(32, 16, 24))
    elif name == "mixed_sph":
        wl = W.mixed_bc_case(n=(16, 48, 32), geometry=W.SPHERICAL, seed=21)
    else:
        return W.by_name(name, n)
    return wl


@pytest.mark.parametrize("name,n", E2E)
def test_nodal_end_to_end_parity(oracle, N, mac, name, n):
    wl = get_case(name, n)
    ref = oracle_project(N, wl)
    K = ref["stats"]["cycles"]
    got = gpu_project(mac, wl)
    if got["stats"]["cycles"] != K:
        got = gpu_project(mac, wl, rel_tol=0.0, max_cycles=K)
    assert got["status"] == ref["status"] == 0
    assert got["stats"]["cycles"] == K
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(got[key], ref[key]) <= E2E_TOL, key
    hg, ho = got["stats"]["res_history"], ref["stats"]["res_history"]
    if hg:
        assert np.allclose(hg, ho[:len(hg)], rtol=1e-3)
        assert hg[-1] <= wl.rel_tol
    assert got["stats"]["rhs_norm_inf"] == pytest.approx(ref["stats"]["rhs_norm_inf"], rel=1e-12)
    assert got["stats"]["rhs_mean_removed"] == pytest.approx(ref["stats"]["rhs_mean_removed"], abs=1e-12 * ref["stats"]["rhs_norm_inf"])
    # node rules on the exported phi
    kind = N.node_kind(ref["g"])
    assert np.all(got["phi"][kind == 1] == 0.0)
    if wl.bc_lo[0] == PER:
        assert np.array_equal(got["phi"][:, :, -1], got["phi"][:, :, 0])


def test_nodal_stop_test_variants_and_edge_cases(oracle, N, mac):
    import torch
    wl = W.config3(N=32, variant="D")
    a, b = gpu_project(mac, wl, stop_test=0), gpu_project(mac, wl, stop_test=1)
    assert a["status"] == b["status"] == 0 and a["stats"]["cycles"] == b["stats"]["cycles"]
    assert a["stats"]["gpu_launches"] < b["stats"]["gpu_launches"]          # the riding test is in use
    for key in ("phi", "u", "v", "w"):
        assert np.array_equal(a[key], b[key]), key
    assert np.allclose(a["stats"]["res_history"], b["stats"]["res_history"], rtol=1e-12)   # the same residual, all unknowns
    # needs desc.nodal = 1
    P = mac.MacProjector(mac.desc_from_workload(wl))
    dv = mac.to_device(wl)
    uc, vc, wc = (tt(x) for x in W.cell_centred(wl))
    rc, _ = P.nodal_project(dv["beta0"], dv["rho0"], dv["rho"], uc, vc, wc, dv["S"], None)
    assert rc == mac.ERR_ARG
    P.close()
    # zero input: nothing to project
    z = W.config1(N=16); z.u[:] = 0; z.v[:] = 0; z.w[:] = 0
    got = gpu_project(mac, z)
    assert got["status"] == 0 and got["stats"]["cycles"] == 0 and np.all(got["u"] == 0)
    # non-finite input
    bad = W.config1(N=16); bad.rho[1, 2, 3] = -1.0
    assert gpu_project(mac, bad)["status"] == mac.ERR_NONFINITE
    # fixed cycle count, unconverged iterate compared with the oracle's
    wl2 = W.config2(N=16)
    tight = dict(bottom_rel_tol=1e-13, bottom_max_iter=2000)
    got = gpu_project(mac, wl2, rel_tol=0.0, max_cycles=3, **tight)
    ref = oracle_project(N, wl2, rel_tol=0.0, max_cycles=3)
    assert got["status"] == 0 and got["stats"]["cycles"] == 3
    assert rel_l2(got["phi"], ref["phi"]) <= E2E_TOL
    assert got["stats"]["res_norm_inf"] == pytest.approx(ref["stats"]["res_norm_inf"], rel=1e-6)
    # the MAC projection and the nodal projection share one handle
    P = mac.MacProjector(mac.desc_from_workload(wl, nodal=1))
    u, v, w = tt(wl.u), tt(wl.v), tt(wl.w)
    rc1, st1 = P.project(dv["beta0"], dv["rho0"], dv["rho"], u, v, w, dv["S"], None)
    rc2, st2 = P.nodal_project(dv["beta0"], dv["rho0"], dv["rho"], uc, vc, wc, dv["S"], None)
    assert rc1 == 0 and rc2 == 0 and st2["cycles"] == a["stats"]["cycles"]
    assert np.array_equal(uc.cpu().numpy(), a["u"])
    P.close()
    torch.cuda.synchronize()
