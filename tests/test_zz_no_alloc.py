"""The allocation-free entry point maestro_mac_lateral_average_noalloc (scratch in a static device array of the
library) against the existing handle path maestro_mac_lateral_average, on two calls in a row.

Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide other tests.
Passes alone in a fresh process (the first call does the per-device set-up) and after the other tests.
"""
import numpy as np
import pytest

from paper_1910_12979_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-13          # the bar of the per-kernel parity tests; the two paths run the same kernels in the same launch
                     # shape with fixed-order sums, so the results are in fact bit-identical (asserted too)


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


def test_noalloc_lateral_average_matches_handle_path_on_two_calls(mac):
    import torch
    # first a large-nr spherical case, then a small planar one: the second call must not see the first one's leftovers
    cases = [W.by_name("4N", 64), W.by_name("2", 32), W.mixed_bc_case(n=(16, 48, 32), geometry=W.SPHERICAL, seed=21)]
    rng = np.random.default_rng(7)
    for rep in range(2):                                   # ... and the whole sequence twice
        for wl in cases:
            rho = tt(wl.rho * (1.0 + 0.1 * rng.standard_normal(wl.rho.shape)))
            desc = mac.desc_from_workload(wl)
            P = mac.MacProjector(desc)
            ref = P.lateral_average(rho).cpu().numpy()     # existing path: scratch in the handle's workspace
            P.close()
            out = torch.full((wl.nr,), float("nan"), dtype=torch.float64, device="cuda")
            assert mac.lateral_average_noalloc(desc, rho, out) == mac.OK
            got = out.cpu().numpy()
            assert np.isfinite(got).all()
            assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
            assert np.array_equal(got, ref)
            out2 = torch.full((wl.nr,), float("nan"), dtype=torch.float64, device="cuda")
            assert mac.lateral_average_noalloc(desc, rho, out2) == mac.OK      # two calls in a row on the same input
            assert np.array_equal(out2.cpu().numpy(), ref)


def test_noalloc_entry_point_allocates_nothing_and_rejects_large_profiles(mac):
    import torch
    wl = W.by_name("3D", 32)
    desc = mac.desc_from_workload(wl)
    rho = tt(wl.rho)
    out = torch.empty(wl.nr, dtype=torch.float64, device="cuda")
    assert mac.lateral_average_noalloc(desc, rho, out) == mac.OK              # (per-device set-up, if this test runs alone)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        assert mac.lateral_average_noalloc(desc, rho, out) == mac.OK
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                                     # no device memory was taken by the calls
    # beyond the static scratch: refused, nothing launched, the output untouched
    big = mac.desc_from_workload(wl, nr=mac.NOALLOC_MAX_NR + 1)
    sentinel = torch.full((mac.NOALLOC_MAX_NR + 1,), -7.0, dtype=torch.float64, device="cuda")
    assert mac.lateral_average_noalloc(big, rho, sentinel) == mac.ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert bool((sentinel == -7.0).all())
    # the largest profile it takes
    edge = mac.desc_from_workload(wl, nr=mac.NOALLOC_MAX_NR, dr=wl.dr * wl.nr / mac.NOALLOC_MAX_NR)
    P = mac.MacProjector(edge)
    ref = P.lateral_average(rho).cpu().numpy()
    P.close()
    oute = torch.empty(mac.NOALLOC_MAX_NR, dtype=torch.float64, device="cuda")
    assert mac.lateral_average_noalloc(edge, rho, oute) == mac.OK
    assert np.array_equal(oute.cpu().numpy(), ref)
    # argument errors
    assert mac.lib().maestro_mac_lateral_average_noalloc(None, None, None, None) == mac.ERR_ARG
