"""Host logic of the launch planners (two-sweep smoother k_rbgs_t2, nodal march k_nod_march) through
maestro_mac_plan_query: pure host arithmetic, no GPU.  Invariants that a wrong wave / chunk decomposition would break:
every tile is covered exactly once, whole-column tiles come in whole waves, the z-chunks of the remaining tiles cover
every plane without an empty chunk, and the block count is what the kernel's index arithmetic expects."""
import itertools

import pytest


@pytest.fixture(scope="module")
def mac():
    from paper_1910_12979_b200 import build, mac
    build.build()
    return mac


def ceil_div(a, b):
    return -(-a // b)


SIZES = [(48, 16, 8), (64, 64, 64), (104, 72, 72), (128, 128, 128), (256, 256, 256), (336, 208, 64), (368, 192, 64),
         (512, 512, 512), (1024, 1024, 1024), (96, 48, 4), (130, 34, 1000), (4096, 18, 16)]
SMS = [1, 2, 108, 132, 148, 160]


@pytest.mark.parametrize("n,sms", list(itertools.product(SIZES, SMS)))
def test_two_sweep_plan_covers_the_level(mac, n, sms):
    nx, ny, nz = n
    p = mac.plan_query(0, nx, ny, nz, sms)
    assert p["tiles_x"] == ceil_div(nx + 1, 26)                      # tile t finishes columns [26 t - 1, 26 t + 25)
    assert p["tiles"] == p["tiles_x"] * ceil_div(ny, 18)
    assert 0 <= p["nfull"] <= p["tiles"] and p["nfull"] % sms == 0   # whole waves of whole-column tiles
    assert p["nsplit"] >= 1 and p["zchunk"] >= 1
    assert p["nsplit"] * p["zchunk"] >= nz                           # the chunks cover every plane ...
    assert (p["nsplit"] - 1) * p["zchunk"] < nz                      # ... and none is empty
    assert p["ncta"] == p["nfull"] + (p["tiles"] - p["nfull"]) * p["nsplit"]
    if p["nfull"] == p["tiles"]:
        assert p["nsplit"] == 1
    if p["nsplit"] > 1:
        assert p["zchunk"] >= 4 or nz < 8                            # chunks of at least 4 planes (each redoes 6)


@pytest.mark.parametrize("n,sms", list(itertools.product(SIZES, SMS)))
def test_nodal_march_plan_covers_the_level(mac, n, sms):
    nx, ny, nz = n
    p = mac.plan_query(1, nx, ny, nz, sms)
    slots = 2 * sms                                                  # two blocks of 256 threads per SM
    assert p["tiles_x"] == ceil_div(nx + 1, 32)
    assert p["tiles"] == p["tiles_x"] * ceil_div(ny + 1, 8)
    assert 0 <= p["nfull"] <= p["tiles"] and p["nfull"] % slots == 0
    assert p["nsplit"] * p["zchunk"] >= nz + 1
    assert (p["nsplit"] - 1) * p["zchunk"] < nz + 1
    assert p["ncta"] == p["nfull"] + (p["tiles"] - p["nfull"]) * p["nsplit"]
    assert p["ncta"] <= 131072                                       # one partial maximum per block (kMaxParts)


def test_bench_size_plans(mac):
    """The decompositions the documented measurements ran (148 SMs)."""
    p = mac.plan_query(0, 512, 512, 512, 148)
    assert (p["tiles"], p["nfull"], p["nsplit"], p["ncta"]) == (580, 0, 1, 580)          # 3.92 waves of whole columns
    p = mac.plan_query(0, 256, 256, 256, 148)
    assert p["tiles"] == 150 and p["nfull"] == 148 and p["nsplit"] > 1                   # one wave + 2 tiles in chunks
    p = mac.plan_query(1, 256, 256, 256, 148)
    assert p["tiles"] == 297 and p["nfull"] == 296 and p["nsplit"] > 1                   # 297 tiles on 296 block slots


def test_plan_query_rejects_bad_arguments(mac):
    import ctypes as C
    info = (C.c_int * 8)()
    L = mac.lib()
    assert L.maestro_mac_plan_query(2, 64, 64, 64, 148, C.byref(info)) == mac.ERR_ARG
    assert L.maestro_mac_plan_query(0, 0, 64, 64, 148, C.byref(info)) == mac.ERR_ARG
    assert L.maestro_mac_plan_query(0, 64, 64, 64, 0, C.byref(info)) == mac.ERR_ARG
    assert L.maestro_mac_plan_query(0, 64, 64, 64, 148, None) == mac.ERR_ARG
