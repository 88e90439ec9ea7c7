"""CPU-side checks of the boundary: libplb.so builds, loads and exports every symbol that
include/plb.h declares; host-only argument checks work; no compute call runs without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def plb():
    from paper_1312_2234_b200 import build, binding
    build.build()
    return binding


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "plb.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"PLB_API\s+[\w\s\*]+?\b(\w+)\s*\(", src)))


def test_header_symbols_are_exported_and_bound(plb):
    names = declared_symbols()
    assert len(names) >= 20 and "lbm_step" in names and "ib_spread" in names
    L = plb.lib()
    for n in names:
        assert hasattr(L, n), "libplb.so does not export %s" % n
        assert n in plb.SYMBOLS, "binding has no signature for %s" % n
    assert sorted(plb.SYMBOLS) == names


def test_north_star_calls_present(plb):
    for n in ("lbm_create", "lbm_set_equilibrium", "ib_add_mesh", "ib_compute_membrane_forces", "ib_spread",
              "lbm_step", "ib_interpolate_advance", "lbm_read_macros"):
        assert n in declared_symbols()


def test_workspace_bytes_host_only(plb):
    n1 = plb.lbm_workspace_bytes(32, 32, 64, 0, 0)
    cells = 32 * 32 * 64
    assert n1 >= 2 * 19 * cells * 4 + 16 * cells   # two fp32 lattices + the (sparsely filled) node-velocity field
    n2 = plb.lbm_workspace_bytes(32, 32, 64, 1000, 3000)
    assert n2 >= n1 + 1000 * (24 + 32) + 3000 * 16
    assert n2 % 256 == 0
    with pytest.raises(plb.PlbError) as e:
        plb.lbm_workspace_bytes(0, 4, 4, 0, 0)
    assert e.value.code == plb.PLB_ERR_ARG
    with pytest.raises(plb.PlbError) as e:
        plb.lbm_workspace_bytes(2048, 2048, 2048, 0, 0)      # >= 2^31 cells
    assert e.value.code == plb.PLB_ERR_ARG and "too large" in str(e.value)


def test_null_context_is_rejected(plb):
    L = plb.lib()
    assert L.lbm_step(None, None) == plb.PLB_ERR_ARG
    assert L.ib_spread(None, None) == plb.PLB_ERR_ARG
    assert L.lbm_destroy(None) == plb.PLB_ERR_ARG
    assert b"null context" in L.plb_last_error()


def test_no_cpu_fallback(plb):
    """Without a CUDA device the product path must fail loudly, not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(plb.PlbError):
        plb.Simulation(8, 8, 8, 0.8)
    # and the raw create call reports a CUDA error, not success
    g = plb.PlbGrid(8, 8, 8)
    b = plb.make_boundary((0, 0, 0))
    h = C.c_void_p()
    fake_ws = C.c_void_p(256 * 1024)
    rc = plb.lib().lbm_create(C.addressof(g), 0.8, C.addressof(b), fake_ws, 1 << 30, 0, 0, None, C.byref(h))
    assert rc == plb.PLB_ERR_CUDA and not h.value


def test_product_does_not_import_oracle():
    """The product path (package, bench's own arm) shares no code with oracle/."""
    pkg = os.path.join(ROOT, "paper_1312_2234_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "orc.h" not in txt and "liboracle" not in txt, f
    orc_c = open(os.path.join(ROOT, "oracle", "orc.c")).read()
    assert "plb" not in orc_c.replace("PLB", "").lower().replace("paper_1312", "")


def test_adhesion_workspace_bytes_host_only(plb):
    n = plb.ib_adhesion_workspace_bytes(64, 32, 48, 1, 10000)       # wall axis y: 64 x 48 vWF sites
    sites = 64 * 48
    # per receptor: node index + (bound, s0, s1, pending site); per site: bond count + lowest pending index
    assert 10000 * (4 + 16) + sites * (4 + 4) <= n <= 10000 * (4 + 16) + sites * (4 + 4) + 4 * 256 and n % 256 == 0
    assert plb.ib_adhesion_workspace_bytes(64, 32, 48, 2, 0) >= 64 * 32 * (4 + 4)
    with pytest.raises(plb.PlbError) as e:
        plb.ib_adhesion_workspace_bytes(64, 32, 48, 3, 10)
    assert e.value.code == plb.PLB_ERR_ARG
    L = plb.lib()
    assert L.ib_adhesion_update(None, 0, 0) == plb.PLB_ERR_ARG
    assert L.ib_set_receptors(None, 0, None, None, None, 0) == plb.PLB_ERR_ARG
