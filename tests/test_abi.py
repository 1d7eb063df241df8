"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol that
include/maestro_mac.h declares, and its descriptor validation / workspace sizing logic works."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mac():
    from paper_1910_12979_b200 import build, mac
    build.build()
    return mac


def test_library_exports_every_declared_symbol(mac):
    hdr = open(os.path.join(ROOT, "include", "maestro_mac.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(maestro_mac_[a-z_]+)\s*\(", hdr))
    assert declared == set(mac.EXPORTS)
    L = mac.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_struct_sizes_match(mac):
    d = mac.Desc()
    mac.lib().maestro_mac_default_desc(C.byref(d))
    assert d.struct_bytes == C.sizeof(mac.Desc)
    assert d.nu_pre == 2 and d.nu_post == 2 and d.rel_tol == 1e-10 and d.coarsest_n == 4


def test_workspace_query_and_validation(mac):
    d = mac.make_desc((128, 128, 128), (1 / 128,) * 3, (0, 0, 1), (0, 0, 1))
    need = mac.workspace_bytes(d)
    # level 0: phi, phi2, rhs + three face arrays; all levels ~ 8/7 of that (+ periodic image columns / rows
    # on the TMA levels, + 2 MB of reduction scratch)
    cells = 128 ** 3
    assert 6 * cells * 8 < need < 8.5 * cells * 8          # (four image columns / rows per side for the two-sweep kernel)
    d2 = mac.make_desc((128, 128, 128), (1 / 128,) * 3, (0, 0, 1), (0, 0, 1), host_staging=1)
    assert mac.workspace_bytes(d2) > need + 6 * cells * 8

    def rc_of(desc):
        need = C.c_size_t(0)
        out = C.c_void_p()
        return mac.lib().maestro_mac_setup(C.byref(desc), None, 0, C.byref(need), C.byref(out))

    bad = mac.make_desc((64, 64, 64), (1 / 64,) * 3, (0, 0, 1), (0, 0, 0))      # periodic on one side
    assert rc_of(bad) == mac.ERR_ARG
    bad = mac.make_desc((64, 0, 64), (1 / 64,) * 3, (0, 0, 1), (0, 0, 1))
    assert rc_of(bad) == mac.ERR_ARG
    bad = mac.make_desc((64, 64, 64), (1 / 64, -1.0, 1 / 64), (0, 0, 1), (0, 0, 1))
    assert rc_of(bad) == mac.ERR_ARG
    bad = mac.make_desc((64, 64, 64), (1 / 64,) * 3, (0, 0, 7), (0, 0, 7))
    assert rc_of(bad) == mac.ERR_ARG
    bad = mac.make_desc((64, 64, 64), (1 / 64,) * 3, (0, 0, 1), (0, 0, 1)); bad.struct_bytes = 8
    assert rc_of(bad) == mac.ERR_ARG
    bad = mac.make_desc((34, 34, 34), (1 / 34,) * 3, (0, 0, 1), (0, 0, 1))      # 17^3 bottom > 4096
    assert rc_of(bad) == mac.ERR_UNSUPPORTED
    bad = mac.make_desc((64, 64, 64), (1 / 64,) * 3, (0, 0, 1), (0, 0, 1), nu_pre=0, nu_post=0)   # no smoothing at all
    assert rc_of(bad) == mac.ERR_ARG
    ok = mac.make_desc((64, 64, 64), (1 / 64,) * 3, (0, 0, 1), (0, 0, 1), nu_pre=0, nu_post=3)    # taken literally
    assert rc_of(ok) == mac.ERR_WORKSPACE
    bad = mac.make_desc((64, 64, 64), (1 / 64,) * 3, (0, 0, 1), (0, 0, 1), timing=2)
    assert rc_of(bad) == mac.ERR_ARG
    assert mac.lib().maestro_mac_setup(None, None, 0, None, None) == mac.ERR_ARG
    assert mac.lib().maestro_mac_status(None, None, None) == mac.ERR_ARG
    assert mac.lib().maestro_mac_level_plan(None, 0, None) == mac.ERR_ARG
    assert mac.lib().maestro_mac_free(None) == mac.OK
    assert mac.lib().maestro_mac_num_levels(None) == mac.ERR_ARG


def test_missing_library_fails_loudly(mac, monkeypatch):
    import paper_1910_12979_b200.mac as m
    monkeypatch.setattr(m, "_lib", None)
    monkeypatch.setattr(m, "LIB_PATH", "/nonexistent/libmaestro_mac.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        m.lib()


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1910_12979_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"mac_oracle|from\s+oracle|import\s+oracle|oracle/", src), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # comments may cite the path
            code = re.sub(r'"""(.|\n)*?"""', "", code)
            assert not re.search(r"maestro_mac|csrc|paper_1910_12979_b200", code), f
