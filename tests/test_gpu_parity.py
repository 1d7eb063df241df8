"""GPU-vs-oracle parity through the C ABI (SURVEY.md Sec. 8(d) "Parity protocol").

Per-kernel parity uses the step API with a 1e-13 relative bar (reading A24: FMA contraction and
evaluation order are not part of the contract); end-to-end parity uses the north_star bar of
1e-10 relative L2 in phi and in u, v, w on the same seeded inputs, with the same cycle count.
"""
import numpy as np
import pytest

from helpers import oracle_project, oracle_structs, rel_l2
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


def tt(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def small_cases():
    return [
        W.mixed_bc_case(n=(16, 8, 12)),
        W.mixed_bc_case(n=(16, 8, 12), geometry=W.SPHERICAL, seed=11),
        W.mixed_bc_case(n=(24, 20, 8), bc_lo=(PER, WALL, OUT), bc_hi=(PER, WALL, WALL), seed=12),
        W.mixed_bc_case(n=(8, 8, 40), bc_lo=(WALL, PER, PER), bc_hi=(OUT, PER, PER), seed=13),
        W.config1(N=16), W.config2(N=16), W.config3(N=16, variant="N"), W.config3(N=16, variant="D"),
        # wide enough for the 64-column TMA tile (x, y not periodic), ragged in x and y, z periodic / not
        W.mixed_bc_case(n=(72, 20, 16), bc_lo=(OUT, WALL, PER), bc_hi=(WALL, OUT, PER), seed=14),
        W.mixed_bc_case(n=(136, 28, 16), bc_lo=(WALL, OUT, OUT), bc_hi=(OUT, WALL, WALL), geometry=W.SPHERICAL, seed=15),
        # wide AND periodic in x and/or y: TMA levels with periodic image columns / rows (ghost layout)
        W.mixed_bc_case(n=(64, 24, 16), bc_lo=(PER, PER, WALL), bc_hi=(PER, PER, OUT), seed=16),
        W.mixed_bc_case(n=(72, 20, 16), bc_lo=(PER, WALL, PER), bc_hi=(PER, OUT, PER), geometry=W.SPHERICAL, seed=17),
        W.mixed_bc_case(n=(120, 16, 16), bc_lo=(OUT, PER, WALL), bc_hi=(OUT, PER, WALL), seed=18),
        W.config1(N=64),
    ]


def folded(O, g, bfaces):
    """internal coefficient a = c_f b / h^2 from the oracle's b (c_f: 1 interior/periodic, 0 WALL, 2 OUTFLOW)."""
    out = []
    for d in range(3):
        a = bfaces[d] / g.h[d] ** 2
        ax = 2 - d
        lo = [slice(None)] * 3; hi = [slice(None)] * 3
        lo[ax] = 0; hi[ax] = a.shape[ax] - 1
        if g.bc_lo[d] != PER:
            a[tuple(lo)] *= 0.0 if g.bc_lo[d] == WALL else 2.0
            a[tuple(hi)] *= 0.0 if g.bc_hi[d] == WALL else 2.0
        out.append(a)
    return out


def close(a, b, tol=KERNEL_TOL):
    a = a.cpu().numpy() if hasattr(a, "cpu") else a
    scale = max(np.abs(b).max(), 1e-300)
    return np.abs(a - b).max() <= tol * scale


@pytest.mark.parametrize("case", range(14))
@pytest.mark.parametrize("smoother", [0, 1, 2, 3, 4])
def test_per_kernel_parity(oracle, mac, case, smoother):
    import torch
    O = oracle
    wl = small_cases()[case]
    g, b, mg = oracle_structs(O, wl)
    # a tight bottom tolerance so that single-V-cycle parity is limited by rounding only
    P = mac.MacProjector(mac.desc_from_workload(wl, smoother=smoother, bottom_rel_tol=1e-13, bottom_max_iter=1000))
    dv = mac.to_device(wl)
    nlev = P.num_levels

    # a2 + a3: coefficients on every level
    P.step_coefficients(dv["beta0"], dv["rho0"], dv["rho"])
    bf = O.face_coeff(g, b, wl.beta0, wl.rho)
    grids, coeffs = [g], [bf]
    while O.can_coarsen(grids[-1], 4):
        gc, cbx, cby, cbz = O.coarsen_coeff(grids[-1], *coeffs[-1])
        grids.append(gc); coeffs.append((cbx, cby, cbz))
    assert nlev == len(grids)
    for l in range(nlev):
        n, h = P.level_dims(l)
        assert list(n) == list(grids[l].n) and np.allclose(h, list(grids[l].h), rtol=1e-15)
        exp = folded(O, grids[l], [c.copy() for c in coeffs[l]])
        for which, e in zip((mac.ARR_BX, mac.ARR_BY, mac.ARR_BZ), exp):
            assert close(P.level_get(l, which), e), (l, which)

    # a4: rhs, its max-norm and the removed mean
    nrm, mean = P.step_rhs(dv["beta0"], dv["u"], dv["v"], dv["w"], dv["S"])
    rhs = O.rhs(g, b, wl.beta0, wl.u, wl.v, wl.w, wl.S)
    m = O.mean(rhs) if O.is_singular(g) else 0.0
    rhs = rhs - m
    assert close(P.level_get(0, mac.ARR_RHS), rhs)
    assert nrm == pytest.approx(np.abs(rhs).max(), rel=1e-12)
    assert mean == pytest.approx(m, abs=1e-13 * np.abs(rhs).max())

    rng = np.random.default_rng(100 + case)
    for l in range(nlev):
        gl, cl = grids[l], coeffs[l]
        shape = O.cell_shape(gl)
        phi = rng.standard_normal(shape)
        f = rng.standard_normal(shape)
        P.level_set(l, mac.ARR_PHI, tt(phi)); P.level_set(l, mac.ARR_RHS, tt(f))
        # a9: residual norm
        assert P.step_residual_norm(l) == pytest.approx(np.abs(O.residual(gl, *cl, phi, f)).max(), rel=1e-12)
        if l + 1 < nlev:
            # a5: two sweeps
            P.step_smooth(l, 2)
            ref = phi.copy(); O.rbgs_sweep(gl, *cl, f, ref); O.rbgs_sweep(gl, *cl, f, ref)
            assert close(P.level_get(l, mac.ARR_PHI), ref), l
            # a6: residual + restriction (and the zeroed coarse phi)
            P.step_residual_restrict(l)
            assert close(P.level_get(l + 1, mac.ARR_RHS), O.restrict(gl, O.residual(gl, *cl, ref, f))), l
            assert float(P.level_get(l + 1, mac.ARR_PHI).abs().max()) == 0.0
            # a7: prolongation
            ec = rng.standard_normal(O.cell_shape(grids[l + 1]))
            P.level_set(l + 1, mac.ARR_PHI, tt(ec))
            P.step_prolong(l)
            O.prolong_add(gl, ec, ref, 0)
            assert close(P.level_get(l, mac.ARR_PHI), ref), l
        else:
            # a8: BiCGStab bottom solve vs the oracle's dense elimination
            P.step_bottom()
            e = O.bottom_solve(gl, *cl, f)
            assert rel_l2(P.level_get(l, mac.ARR_PHI).cpu().numpy(), e) <= 1e-9

    # one whole V-cycle from a random state on level 0
    phi = rng.standard_normal(O.cell_shape(g)); f = rng.standard_normal(O.cell_shape(g))
    if O.is_singular(g):
        f -= f.mean()
    P.level_set(0, mac.ARR_PHI, tt(phi)); P.level_set(0, mac.ARR_RHS, tt(f))
    P.step_vcycle()
    ref = phi.copy(); O.vcycle(g, *bf, f, ref, mg)
    assert rel_l2(P.level_get(0, mac.ARR_PHI).cpu().numpy(), ref) <= 1e-9

    # a10: correction from a given phi
    P.level_set(0, mac.ARR_PHI, tt(phi))
    u, v, w = tt(wl.u), tt(wl.v), tt(wl.w)
    P.step_correct(dv["rho0"], dv["rho"], u, v, w)
    ru, rv, rw = wl.u.copy(), wl.v.copy(), wl.w.copy()
    O.correct(g, wl.rho, phi, ru, rv, rw)
    assert close(u, ru) and close(v, rv) and close(w, rw)
    torch.cuda.synchronize()
    P.close()


E2E_CASES = [("1", 32), ("2", 32), ("3N", 32), ("3D", 32), ("4N", 32), ("4D", 64), ("5", 32),
             ("2", 64), ("3N", 64), ("mixed", 0), ("mixed_sph", 0), ("1", 64), ("5", 128), ("wide_bottom", 0)]


def get_case(name, N):
    if name == "mixed":
        return W.mixed_bc_case(n=(32, 16, 24))
    if name == "wide_bottom":    # the coarsest level (64 x 8 x 4, periodic in x) is as wide as a TMA level: it keeps the plain layout
        wl = W.mixed_bc_case(n=(128, 16, 8), bc_lo=(PER, WALL, OUT), bc_hi=(PER, WALL, WALL), seed=22)
        wl.dx = (1.0 / 128,) * 3          # cubic cells (point Gauss-Seidel does not like the 20:1 boxes of the recipe)
        wl.dr = wl.dx[2]
        return wl
    if name == "mixed_sph":
        return W.mixed_bc_case(n=(16, 48, 32), geometry=W.SPHERICAL, seed=21)
    return W.by_name(name, N)


def gpu_project(mac, wl, **over):
    import torch
    P = mac.MacProjector(mac.desc_from_workload(wl, **over))
    dv = mac.to_device(wl)
    phi = torch.full((wl.n[2], wl.n[1], wl.n[0]), float("nan"), dtype=torch.float64, device="cuda")
    rc, st = P.project(dv["beta0"], dv["rho0"], dv["rho"], dv["u"], dv["v"], dv["w"], dv["S"], phi)
    out = dict(status=rc, stats=st, phi=phi.cpu().numpy(), u=dv["u"].cpu().numpy(),
               v=dv["v"].cpu().numpy(), w=dv["w"].cpu().numpy())
    P.close()
    return out


@pytest.mark.parametrize("name,N", E2E_CASES)
@pytest.mark.parametrize("smoother", [0, 1, 2, 3, 4])
def test_end_to_end_parity(oracle, mac, name, N, smoother):
    O = oracle
    wl = get_case(name, N)
    ref = oracle_project(O, wl)
    K = ref["stats"]["cycles"]
    got = gpu_project(mac, wl, smoother=smoother)
    if got["stats"]["cycles"] != K:            # knife-edge on the stop test: rerun in lockstep
        got = gpu_project(mac, wl, smoother=smoother, rel_tol=0.0, max_cycles=K)
    assert got["status"] == ref["status"] == 0
    assert got["stats"]["cycles"] == K
    assert got["stats"]["singular"] == ref["stats"]["singular"]
    assert got["stats"]["levels"] == ref["stats"]["levels"]
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(got[key], ref[key]) <= E2E_TOL, key
    # same residual reduction
    hist_g, hist_o = got["stats"]["res_history"], ref["stats"]["res_history"]
    if hist_g:
        assert np.allclose(hist_g, hist_o[:len(hist_g)], rtol=1e-3)
        assert hist_g[-1] <= wl.rel_tol
    assert got["stats"]["rhs_norm_inf"] == pytest.approx(ref["stats"]["rhs_norm_inf"], rel=1e-12)
    assert got["stats"]["rhs_mean_removed"] == pytest.approx(ref["stats"]["rhs_mean_removed"], abs=1e-12 * ref["stats"]["rhs_norm_inf"])
    # the paper's constraint (Eq. 6) holds for the GPU result, checked with the oracle's operator
    c = O.constraint(ref["g"], ref["b"], wl.beta0, got["u"], got["v"], got["w"], wl.S) - ref["stats"]["rhs_mean_removed"]
    assert np.abs(c).max() <= wl.rel_tol * ref["stats"]["rhs_norm_inf"] * 1.01


def test_edge_cases(oracle, mac):
    import torch
    O = oracle
    # rhs == 0: OK, cycles 0, phi 0, velocities untouched
    z = W.config1(N=8); z.u[:] = 0; z.v[:] = 0; z.w[:] = 0
    got = gpu_project(mac, z)
    assert got["status"] == 0 and got["stats"]["cycles"] == 0 and np.all(got["phi"] == 0) and np.all(got["u"] == 0)
    # non-finite inputs
    bad = W.config1(N=8); bad.u[1, 2, 3] = np.nan
    assert gpu_project(mac, bad)["status"] == mac.ERR_NONFINITE
    bad = W.config1(N=8); bad.rho[0, 0, 0] = -1.0
    assert gpu_project(mac, bad)["status"] == mac.ERR_NONFINITE
    # max_cycles reached: NOT_CONVERGED with the last iterate written, same as the oracle's
    wl = W.config2(N=16)
    # (an unconverged iterate is compared, so the inexact bottom solve is not yet contracted away:
    # use a tight BiCGStab tolerance)
    tight = dict(bottom_rel_tol=1e-13, bottom_max_iter=1000)
    got = gpu_project(mac, wl, max_cycles=2, **tight)
    ref = oracle_project(O, wl, max_cycles=2)
    assert got["status"] == mac.NOT_CONVERGED and ref["status"] == 1
    assert rel_l2(got["phi"], ref["phi"]) <= E2E_TOL and rel_l2(got["w"], ref["w"]) <= E2E_TOL
    # rel_tol = 0: exactly max_cycles cycles
    got = gpu_project(mac, wl, rel_tol=0.0, max_cycles=3, **tight)
    ref = oracle_project(O, wl, rel_tol=0.0, max_cycles=3)
    assert got["status"] == 0 and got["stats"]["cycles"] == 3
    assert rel_l2(got["phi"], ref["phi"]) <= E2E_TOL
    assert got["stats"]["res_norm_inf"] == pytest.approx(ref["stats"]["res_norm_inf"], rel=1e-6)
    # rho == NULL (base-state-only projection), S == NULL, phi == NULL
    P = mac.MacProjector(mac.desc_from_workload(wl))
    dv = mac.to_device(wl)
    rc, st = P.project(dv["beta0"], dv["rho0"], None, dv["u"], dv["v"], dv["w"], None, None)
    g, b, mg = oracle_structs(O, wl)
    u, v, w = wl.u.copy(), wl.v.copy(), wl.w.copy()
    ost, _, ostats = O.project(g, b, mg, wl.beta0, wl.rho0, None, u, v, w, None)
    assert rc == ost == 0 and st["cycles"] == ostats["cycles"]
    assert rel_l2(dv["u"].cpu().numpy(), u) <= E2E_TOL and rel_l2(dv["w"].cpu().numpy(), w) <= E2E_TOL
    # argument errors
    rc, _ = P.project(None, dv["rho0"], dv["rho"], dv["u"], dv["v"], dv["w"])
    assert rc == mac.ERR_ARG
    rc, _ = P.project(dv["beta0"], dv["rho0"], dv["rho"], dv["u"], dv["u"], dv["w"])
    assert rc == mac.ERR_ARG
    rc, _ = P.project_host(dv["beta0"], dv["rho0"], dv["rho"], dv["u"], dv["v"], dv["w"])
    assert rc == mac.ERR_ARG                      # no staging reserved
    P.close()
    # a single-level problem (level 0 is the bottom): BiCGStab alone must solve it
    tiny = W.mixed_bc_case(n=(6, 5, 7), bc_lo=(OUT, WALL, WALL), bc_hi=(WALL, OUT, WALL))
    got = gpu_project(mac, tiny, bottom_rel_tol=1e-13, bottom_max_iter=500)
    ref = oracle_project(O, tiny)
    assert ref["stats"]["levels"] == 1 and got["stats"]["levels"] == 1
    assert rel_l2(got["phi"], ref["phi"]) <= 1e-8
    torch.cuda.synchronize()


def test_project_host_matches_device_path(oracle, mac):
    import torch
    wl = W.config3(N=32, variant="D")
    ref = gpu_project(mac, wl)
    P = mac.MacProjector(mac.desc_from_workload(wl, host_staging=1))
    pin = lambda a: torch.from_numpy(a.copy()).pin_memory()
    u, v, w, phi = pin(wl.u), pin(wl.v), pin(wl.w), torch.empty(wl.rho.shape, dtype=torch.float64).pin_memory()
    rc, st = P.project_host(pin(wl.beta0), pin(wl.rho0), pin(wl.rho), u, v, w, pin(wl.S), phi)
    assert rc == 0 and st["cycles"] == ref["stats"]["cycles"]
    assert np.array_equal(phi.numpy(), ref["phi"]) and np.array_equal(u.numpy(), ref["u"])
    assert np.array_equal(w.numpy(), ref["w"])
    P.close()


@pytest.mark.parametrize("nset", [2, 3])
def test_project_host_seq_pipelined(oracle, mac, nset):
    """maestro_mac_project_host_seq (config 5's pattern: consecutive projections with a new U_edge each step, transfers
    overlapped with the neighbouring steps): every step equals the one-at-a-time call bit for bit, with in-place and
    separate output buffers, and the oracle on the step's own U_edge."""
    import torch
    steps = [W.config5(N=64, step=k) for k in range(5)]
    wl = steps[0]
    pin = lambda a: torch.from_numpy(a.copy()).pin_memory()
    P = mac.MacProjector(mac.desc_from_workload(wl, host_staging=nset))
    one = []
    for sw in steps:                               # references: the single call, one step at a time
        u, v, w, phi = pin(sw.u), pin(sw.v), pin(sw.w), torch.empty(wl.rho.shape, dtype=torch.float64).pin_memory()
        rc, st = P.project_host(pin(wl.beta0), pin(wl.rho0), pin(wl.rho), u, v, w, pin(wl.S), phi)
        assert rc == 0
        one.append((u.numpy().copy(), v.numpy().copy(), w.numpy().copy(), phi.numpy().copy(), st["cycles"]))
    ui, vi, wi = [pin(sw.u) for sw in steps], [pin(sw.v) for sw in steps], [pin(sw.w) for sw in steps]
    uo = [torch.empty_like(t).pin_memory() for t in ui]
    phis = [torch.empty(wl.rho.shape, dtype=torch.float64).pin_memory() for _ in steps]
    # u in place, v and w into separate buffers (two of them, reused every other step, as bench.py does: checked at the end)
    vo2, wo2 = [torch.empty_like(vi[0]).pin_memory() for _ in range(2)], [torch.empty_like(wi[0]).pin_memory() for _ in range(2)]
    rc, sts = P.project_host_seq(pin(wl.beta0), pin(wl.rho0), pin(wl.rho), pin(wl.S), ui, vi, wi, ui,
                                 [vo2[k & 1] for k in range(5)], [wo2[k & 1] for k in range(5)], phis)
    assert rc == 0 and [st["cycles"] for st in sts] == [o[4] for o in one]
    for k in range(5):
        assert np.array_equal(ui[k].numpy(), one[k][0]) and np.array_equal(phis[k].numpy(), one[k][3]), k
    for k in (3, 4):                               # the last writers of the two rotating buffers
        assert np.array_equal(vo2[k & 1].numpy(), one[k][1]) and np.array_equal(wo2[k & 1].numpy(), one[k][2]), k
    ref = oracle_project(oracle, steps[4])
    assert ref["stats"]["cycles"] == one[4][4]
    assert rel_l2(one[4][0], ref["u"]) <= E2E_TOL and rel_l2(one[4][3], ref["phi"]) <= E2E_TOL
    # separate outputs for everything, inputs untouched
    rc, sts = P.project_host_seq(pin(wl.beta0), pin(wl.rho0), pin(wl.rho), pin(wl.S), [pin(sw.u) for sw in steps[:2]],
                                 vi[:2], wi[:2], uo[:2], [vo2[0], vo2[1]], [wo2[0], wo2[1]], None)
    assert rc == 0
    for k in range(2):
        assert np.array_equal(uo[k].numpy(), one[k][0]) and np.array_equal(vo2[k].numpy(), one[k][1]), k
        assert np.array_equal(vi[k].numpy(), steps[k].v)
    # argument errors: no double staging; a NULL step pointer
    rc, _ = P.project_host_seq(pin(wl.beta0), pin(wl.rho0), pin(wl.rho), pin(wl.S), [ui[0]], [vi[0]], [None], [ui[0]], [vo2[0]], [wo2[0]])
    assert rc == mac.ERR_ARG
    P.close()
    P1 = mac.MacProjector(mac.desc_from_workload(wl, host_staging=1))
    rc, _ = P1.project_host_seq(pin(wl.beta0), pin(wl.rho0), pin(wl.rho), pin(wl.S), [ui[0]], [vi[0]], [wi[0]], [uo[0]], [vo2[0]], [wo2[0]])
    assert rc == mac.ERR_ARG
    P1.close()


@pytest.mark.parametrize("name,N", [("1", 32), ("2", 32), ("3D", 32), ("3N", 16)])
def test_device_side_solve_of_small_problems(oracle, mac, name, N):
    """A problem whose level 0 has at most 32^3 cells is solved by ONE launch of k_cluster_vcycles (cycles and stop test
    on the device): same cycle count and residual history as the host-driven solve of
    smoother 4 (one launch per step, k_coarse_tail, stop test read by the host every cycle), results equal up to the
    bottom solver's rounding (one-warp BiCGStab there, block BiCGStab here), a handful of launches, and the oracle's result."""
    wl = W.by_name(name, N)
    P = mac.MacProjector(mac.desc_from_workload(wl))
    assert P.level_plan(0)["kernel"] == "cluster", P.level_plan(0)
    P.close()
    a, b = gpu_project(mac, wl), gpu_project(mac, wl, smoother=4)
    assert a["status"] == b["status"] == 0 and a["stats"]["cycles"] == b["stats"]["cycles"]
    assert a["stats"]["gpu_launches"] <= 20 < b["stats"]["gpu_launches"]
    assert np.allclose(a["stats"]["res_history"], b["stats"]["res_history"], rtol=1e-6)
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(a[key], b[key]) <= 1e-12, key
    ref = oracle_project(oracle, wl)
    assert ref["stats"]["cycles"] == a["stats"]["cycles"]
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(a[key], ref[key]) <= E2E_TOL, key
    # fixed cycle count: the history is filled, the final norm reported
    c = gpu_project(mac, wl, rel_tol=0.0, max_cycles=3)
    assert c["status"] == 0 and c["stats"]["cycles"] == 3
    assert np.allclose(c["stats"]["res_history"], a["stats"]["res_history"][:3], rtol=1e-12)


def test_asynchronous_fixed_cycle_call(oracle, mac):
    """rel_tol = 0 and stats = NULL: the call returns without synchronising; maestro_mac_status() completes it with
    the same results and stats as the synchronous fixed-cycle call, and reports non-finite input."""
    import torch
    wl = W.config2(N=32)
    ref = gpu_project(mac, wl, rel_tol=0.0, max_cycles=4)
    P = mac.MacProjector(mac.desc_from_workload(wl, rel_tol=0.0, max_cycles=4))
    dv = mac.to_device(wl)
    phi = torch.empty(wl.rho.shape, dtype=torch.float64, device="cuda")
    rc, st = P.project(dv["beta0"], dv["rho0"], dv["rho"], dv["u"], dv["v"], dv["w"], dv["S"], phi, want_stats=False)
    assert rc == 0 and st is None
    rc, st = P.status()
    assert rc == 0 and st["cycles"] == 4
    assert st["rhs_norm_inf"] == ref["stats"]["rhs_norm_inf"]
    # (the synchronous call of a problem this small takes the norm inside k_cluster_vcycles, status() by k_residual_norm)
    assert st["res_norm_inf"] == pytest.approx(ref["stats"]["res_norm_inf"], rel=1e-9)
    assert np.array_equal(phi.cpu().numpy(), ref["phi"]) and np.array_equal(dv["u"].cpu().numpy(), ref["u"])
    rc2, st2 = P.status()                          # idempotent: the stats of the last call, no work
    assert rc2 == 0 and st2["cycles"] == 4
    # zero rhs: the cycles run on zeros, the velocities stay bit for bit
    z = W.config1(N=16); z.u[:] = 0; z.v[:] = 0; z.w[:] = 0; z.u[3, 4, 5] = -0.0
    Pz = mac.MacProjector(mac.desc_from_workload(z, rel_tol=0.0, max_cycles=2))
    dz = mac.to_device(z)
    phiz = torch.full(z.rho.shape, float("nan"), dtype=torch.float64, device="cuda")
    rc, _ = Pz.project(dz["beta0"], dz["rho0"], dz["rho"], dz["u"], dz["v"], dz["w"], None, phiz, want_stats=False)
    assert rc == 0 and Pz.status(want_stats=False)[0] == 0
    assert float(phiz.abs().max()) == 0.0 and np.array_equal(dz["u"].cpu().numpy(), z.u)
    Pz.close()
    # non-finite input surfaces in maestro_mac_status
    bad = W.config2(N=32); bad.rho[1, 2, 3] = -1.0
    db = mac.to_device(bad)
    rc, _ = P.project(db["beta0"], db["rho0"], db["rho"], db["u"], db["v"], db["w"], db["S"], None, want_stats=False)
    assert rc == 0
    assert P.status()[0] == mac.ERR_NONFINITE
    P.close()


def test_per_launch_timing_is_opt_in(mac):
    wl = W.config3(N=64, variant="D")
    off, on = gpu_project(mac, wl), gpu_project(mac, wl, timing=1)
    assert off["stats"]["smooth0_timed"] == 0 and off["stats"]["ms_smooth0"] == 0.0
    assert off["stats"]["smooth0_launches"] == on["stats"]["smooth0_launches"] > 0
    assert on["stats"]["smooth0_timed"] == on["stats"]["smooth0_launches"] and on["stats"]["ms_smooth0"] > 0.0
    assert np.array_equal(off["phi"], on["phi"])


def test_deterministic_across_runs(mac):
    wl = W.config2(N=32)
    a, b = gpu_project(mac, wl), gpu_project(mac, wl)
    for key in ("phi", "u", "v", "w"):
        assert np.array_equal(a[key], b[key])


@pytest.mark.parametrize("name,N", [("4D", 64), ("3N", 64), ("mixed_wide", 0)])
def test_stop_test_riding_on_the_next_sweep(oracle, mac, name, N):
    """stop_test 0 (red-cell residual from the next cycle's first pre-sweep) and 1 (separate kernel over all
    cells) take the same decisions and leave bit-identical results: the speculative sweep is either the next
    cycle's first pre-sweep or dropped."""
    wl = (W.mixed_bc_case(n=(128, 80, 96), bc_lo=(WALL, OUT, OUT), bc_hi=(OUT, WALL, WALL), geometry=W.SPHERICAL, seed=15)
          if name == "mixed_wide" else W.by_name(name, N))
    a, b = gpu_project(mac, wl, stop_test=0), gpu_project(mac, wl, stop_test=1)
    assert a["status"] == b["status"] == 0
    assert a["stats"]["cycles"] == b["stats"]["cycles"]
    assert a["stats"]["gpu_launches"] < b["stats"]["gpu_launches"]        # the riding test is actually in use
    for key in ("phi", "u", "v", "w"):
        assert np.array_equal(a[key], b[key]), key
    # black residuals are at rounding level after a post-sweep: the two norms agree far above it
    assert np.allclose(a["stats"]["res_history"], b["stats"]["res_history"], rtol=1e-4)
    ref = oracle_project(oracle, wl)
    assert ref["stats"]["cycles"] == a["stats"]["cycles"]
    assert np.allclose(a["stats"]["res_history"], ref["stats"]["res_history"], rtol=1e-3)


T2_CASES = [
    dict(n=(104, 72, 72), bc_lo=(WALL, OUT, OUT), bc_hi=(OUT, WALL, WALL), geometry=W.SPHERICAL, seed=31),
    dict(n=(96, 48, 64), bc_lo=(PER, PER, PER), bc_hi=(PER, PER, PER), seed=32),
    dict(n=(64, 80, 40), bc_lo=(OUT, PER, WALL), bc_hi=(WALL, PER, OUT), seed=33),
    dict(n=(128, 16, 8), bc_lo=(PER, WALL, PER), bc_hi=(PER, WALL, PER), seed=34),
]


@pytest.mark.parametrize("case", range(len(T2_CASES)))
def test_two_sweep_kernel_equals_two_single_sweeps(oracle, mac, case):
    """k_rbgs_t2 (two sweeps per pass, smoother 0) is bit-identical to two launches of the single-sweep TMA kernel
    (smoother 4) and matches two oracle sweeps; sizes span several tiles, a ragged tail and several z-chunks."""
    O = oracle
    wl = W.mixed_bc_case(**T2_CASES[case])
    g, b, mg = oracle_structs(O, wl)
    dv = mac.to_device(wl)
    rng = np.random.default_rng(200 + case)
    phi = rng.standard_normal(O.cell_shape(g)); f = rng.standard_normal(O.cell_shape(g))
    bf = O.face_coeff(g, b, wl.beta0, wl.rho)
    got = {}
    for sm in (0, 4):
        P = mac.MacProjector(mac.desc_from_workload(wl, smoother=sm))
        P.step_coefficients(dv["beta0"], dv["rho0"], dv["rho"])
        P.level_set(0, mac.ARR_PHI, tt(phi)); P.level_set(0, mac.ARR_RHS, tt(f))
        P.step_smooth(0, 2)
        got[sm, 2] = P.level_get(0, mac.ARR_PHI).cpu().numpy()
        P.step_smooth(0, 3)                       # a pair and a single sweep
        got[sm, 5] = P.level_get(0, mac.ARR_PHI).cpu().numpy()
        P.close()
    assert np.array_equal(got[0, 2], got[4, 2])
    assert np.array_equal(got[0, 5], got[4, 5])
    ref = phi.copy(); O.rbgs_sweep(g, *bf, f, ref); O.rbgs_sweep(g, *bf, f, ref)
    assert close(got[4, 2], ref)


@pytest.mark.parametrize("name,N,smoother", [("2", 32, 0), ("3D", 32, 0), ("4N", 32, 1), ("mixed_sph", 0, 2), ("wide_bottom", 0, 0)])
def test_harmonic_face_density_variant(oracle, mac, name, N, smoother):
    """desc.rho_mean = 1 (reading A3, harmonic variant): coefficients, correction and the whole projection match the
    oracle run with the same flag."""
    O = oracle
    wl = get_case(name, N)
    wl.meta["rho_mean"] = 1
    g, b, mg = oracle_structs(O, wl)
    P = mac.MacProjector(mac.desc_from_workload(wl, smoother=smoother))
    dv = mac.to_device(wl)
    P.step_coefficients(dv["beta0"], dv["rho0"], dv["rho"])
    exp = folded(O, g, [c.copy() for c in O.face_coeff(g, b, wl.beta0, wl.rho)])
    for which, e in zip((mac.ARR_BX, mac.ARR_BY, mac.ARR_BZ), exp):
        assert close(P.level_get(0, which), e), which
    rng = np.random.default_rng(3)
    phi = rng.standard_normal(O.cell_shape(g))
    P.level_set(0, mac.ARR_PHI, tt(phi))
    u, v, w = tt(wl.u), tt(wl.v), tt(wl.w)
    P.step_correct(dv["rho0"], dv["rho"], u, v, w)
    ru, rv, rw = wl.u.copy(), wl.v.copy(), wl.w.copy()
    O.correct(g, wl.rho, phi, ru, rv, rw)
    assert close(u, ru) and close(v, rv) and close(w, rw)
    P.close()
    ref = oracle_project(O, wl)
    got = gpu_project(mac, wl, smoother=smoother)
    if got["stats"]["cycles"] != ref["stats"]["cycles"]:
        got = gpu_project(mac, wl, smoother=smoother, rel_tol=0.0, max_cycles=ref["stats"]["cycles"])
    assert got["status"] == ref["status"] == 0 and got["stats"]["cycles"] == ref["stats"]["cycles"]
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(got[key], ref[key]) <= E2E_TOL, key


@pytest.mark.parametrize("nu_pre,nu_post", [(1, 1), (3, 1), (1, 2), (4, 3), (0, 3), (2, 0)])
@pytest.mark.parametrize("name,N", [("1", 64), ("4D", 64)])
def test_sweep_counts_other_than_two(oracle, mac, name, N, nu_pre, nu_post):
    """Pairs of sweeps run through the two-sweep kernel, a remaining one through the single-sweep kernel, and the
    riding stop test follows (one- or two-sweep speculative pass): parity for odd and larger sweep counts."""
    wl = W.by_name(name, N)
    wl.nu_pre, wl.nu_post = nu_pre, nu_post
    ref = oracle_project(oracle, wl)
    K = ref["stats"]["cycles"]
    got = gpu_project(mac, wl)
    if got["stats"]["cycles"] != K:
        got = gpu_project(mac, wl, rel_tol=0.0, max_cycles=K)
    assert got["status"] == ref["status"] == 0 and got["stats"]["cycles"] == K
    for key in ("phi", "u", "v", "w"):
        assert rel_l2(got[key], ref[key]) <= E2E_TOL, key
