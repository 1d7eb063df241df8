"""GPU-vs-oracle parity of the base-state steps: beta0 from p0 and Gamma1bar
(Eq. 5), the dp0/dt term of the constraint (Eq. 6) in the rhs kernel, and a whole
projection with both, through the C ABI."""
import numpy as np
import pytest

from helpers import oracle_structs, rel_l2
from paper_1910_12979_b200 import workloads as W
from test_gpu_parity import E2E_TOL, KERNEL_TOL, close, tt

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mac():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_12979_b200 import build, mac
    build.build()
    return mac


@pytest.mark.parametrize("nr", [1, 2, 31, 32, 33, 887, 4099])
def test_base_state_kernel_matches_oracle(oracle, mac, nr):
    rng = np.random.default_rng(nr)
    r = (np.arange(nr) + 0.5) / nr
    rho0 = np.exp(-r / 0.2) * (1 + 0.01 * rng.standard_normal(nr))
    p0 = rho0 ** (5 / 3) * np.exp(0.05 * rng.standard_normal(nr))
    gam = rng.uniform(1.2, 1.7, nr)
    dpdt = rng.uniform(-1, 1, nr)
    beta0, q = mac.base_state(tt(rho0), tt(p0), tt(gam), tt(dpdt))
    assert close(beta0, oracle.make_beta0(rho0, p0, gam), 1e-12)       # a running sum of nr terms
    assert close(q, oracle.dpdt_term(p0, gam, dpdt))
    beta0_only, none = mac.base_state(tt(rho0), tt(p0), tt(gam))
    assert none is None and np.array_equal(beta0_only.cpu().numpy(), beta0.cpu().numpy())


CASES = [("2", 32, 0), ("3D", 32, 0), ("3N", 32, 1), ("mixed_sph", 0, 2), ("1", 64, 0)]


@pytest.mark.parametrize("name,N,smoother", CASES)
def test_rhs_and_projection_with_dpdt_term(oracle, mac, name, N, smoother):
    O = oracle
    wl = W.mixed_bc_case(n=(16, 48, 32), geometry=W.SPHERICAL, seed=21) if name == "mixed_sph" else W.by_name(name, N)
    wl = W.with_base_state(wl)
    g, b, mg = oracle_structs(O, wl)
    p0, gam, dpdt = wl.meta["p0"], wl.meta["gamma1bar"], wl.meta["dp0dt"]
    # oracle: Eq. 5, Eq. 6 term, effective source, then the usual projection
    beta0 = O.make_beta0(wl.rho0, p0, gam)
    q = O.dpdt_term(p0, gam, dpdt)
    S_eff = O.effective_source(g, b, wl.S, q)
    u, v, w = wl.u.copy(), wl.v.copy(), wl.w.copy()
    ost, ophi, ostats = O.project(g, b, mg, beta0, wl.rho0, wl.rho, u, v, w, S_eff)
    # CUDA path: base-state kernel, registered term, rhs kernel, whole projection
    dv = mac.to_device(wl)
    d_beta0, d_q = mac.base_state(dv["rho0"], tt(p0), tt(gam), tt(dpdt))
    P = mac.MacProjector(mac.desc_from_workload(wl, smoother=smoother))
    P.set_dpdt_term(d_q)
    nrm, mean = P.step_rhs(d_beta0, dv["u"], dv["v"], dv["w"], dv["S"])
    rhs = O.rhs(g, b, beta0, wl.u, wl.v, wl.w, S_eff)
    m = O.mean(rhs) if O.is_singular(g) else 0.0
    assert close(P.level_get(0, mac.ARR_RHS), rhs - m)
    assert nrm == pytest.approx(np.abs(rhs - m).max(), rel=1e-12)
    import torch
    phi = torch.empty(wl.rho.shape, dtype=torch.float64, device="cuda")
    rc, st = P.project(d_beta0, dv["rho0"], dv["rho"], dv["u"], dv["v"], dv["w"], dv["S"], phi)
    if st["cycles"] != ostats["cycles"]:                       # knife-edge on the stop test: lockstep rerun
        P.close()
        dv = mac.to_device(wl)
        P = mac.MacProjector(mac.desc_from_workload(wl, smoother=smoother, rel_tol=0.0, max_cycles=ostats["cycles"]))
        P.set_dpdt_term(d_q)
        rc, st = P.project(d_beta0, dv["rho0"], dv["rho"], dv["u"], dv["v"], dv["w"], dv["S"], phi)
    assert rc == ost == 0 and st["cycles"] == ostats["cycles"]
    assert rel_l2(phi.cpu().numpy(), ophi) <= E2E_TOL
    for key, ref in (("u", u), ("v", v), ("w", w)):
        assert rel_l2(dv[key].cpu().numpy(), ref) <= E2E_TOL, key
    # the constraint of Eq. 6 with its dp0/dt term, evaluated by the oracle's operators on the GPU result
    c = O.constraint(g, b, beta0, dv["u"].cpu().numpy(), dv["v"].cpu().numpy(), dv["w"].cpu().numpy(), S_eff) - ostats["rhs_mean_removed"]
    assert np.abs(c).max() <= wl.rel_tol * ostats["rhs_norm_inf"] * 1.01
    # clearing the term restores the plain rhs
    P.set_dpdt_term(None)
    P.step_rhs(d_beta0, tt(wl.u), tt(wl.v), tt(wl.w), dv["S"])
    rhs0 = O.rhs(g, b, beta0, wl.u, wl.v, wl.w, wl.S)
    assert close(P.level_get(0, mac.ARR_RHS), rhs0 - (O.mean(rhs0) if O.is_singular(g) else 0.0))
    P.close()


@pytest.mark.parametrize("name,N", [("2", 32), ("3D", 32), ("mixed_sph", 0), ("5", 64), ("4N", 64)])
def test_lateral_average_matches_oracle(oracle, mac, name, N):
    """maestro_mac_lateral_average vs oracle O13: every cell lands in the same sample on both sides
    (the binning arithmetic is the oracle's, operation by operation), so the means agree to the order of additions
    and the filled samples to rounding."""
    wl = W.mixed_bc_case(n=(16, 48, 32), geometry=W.SPHERICAL, seed=21) if name == "mixed_sph" else W.by_name(name, N)
    g, b, _ = oracle_structs(oracle, wl)
    ref, cnt = oracle.lateral_average(g, b, wl.rho)
    P = mac.MacProjector(mac.desc_from_workload(wl))
    got = P.lateral_average(tt(wl.rho)).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    for _ in range(3):                                            # fixed-order sums: bit-reproducible from run to run
        again = P.lateral_average(tt(wl.rho)).cpu().numpy()
        assert np.array_equal(again, got)
    P.close()
